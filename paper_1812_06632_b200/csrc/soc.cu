// libsoc_b200 -- photon-package simulation and temperature kernels for sm_100a, plus the C ABI of
// include/soc.h.  See DESIGN.md for the data layout, the kernels and the rooflines that bound them.
//
// No tensor cores here: the path is a random walk with one dependent 4-byte gather and one 8-byte
// scatter-add per cell-step, not a dense contraction (BASELINE.json:north_star).
#include "soc.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

// ------------------------------------------------------------------------------------------------
// host-side bookkeeping
// ------------------------------------------------------------------------------------------------
namespace {

thread_local std::string g_last_error;
unsigned long long g_launches = 0;

// process-wide cache of the package-queue buffers of slab-blocked launches (see soc_release_cached_memory in soc.h)
struct CachedBuffer { void *ptr; size_t entries; int device; };
std::vector<CachedBuffer> g_queue_cache;
std::mutex g_queue_cache_mutex;
constexpr size_t kQueueCacheMax = 2;

// ... and of the large per-grid arrays (cell words, links, accumulators): soc_run_host creates and destroys a grid per call,
// and cudaMalloc / cudaFree of a dozen buffers of 45-140 MB cost it 10-80 ms, differently every time.  big_malloc takes a
// cached buffer of exactly the size asked for if there is one; big_free hands buffers of >= 1 MB to the cache (at most
// big_cache_limit() in total), the others to cudaFree.  A cudaMalloc that fails empties both caches and is tried again.  Contents are undefined, as after cudaMalloc.
struct BigBuffer { void *ptr; size_t bytes; int device; };
std::vector<BigBuffer> g_big_cache, g_big_live;
std::mutex g_big_mutex;
// most the big cache keeps, in bytes: 8 GB, or SOC_B200_CACHE_MB megabytes from the environment (0 = keep nothing)
size_t big_cache_limit()
{
    static const size_t limit = [] {
        const char *v = std::getenv("SOC_B200_CACHE_MB");
        char *end = nullptr;
        const unsigned long long mb = v ? std::strtoull(v, &end, 10) : 0;
        return v && end != v ? (size_t)mb << 20 : (size_t)8 << 30;
    }();
    return limit;
}

int64_t release_caches();           // frees both caches (device synchronised); the caller holds neither mutex

cudaError_t big_malloc_impl(void **out, size_t bytes)
{
    int device = 0;
    cudaGetDevice(&device);
    {
        std::lock_guard<std::mutex> lock(g_big_mutex);
        for (size_t i = 0; i < g_big_cache.size(); ++i)
            if (g_big_cache[i].bytes == bytes && g_big_cache[i].device == device) {
                *out = g_big_cache[i].ptr;
                g_big_live.push_back(g_big_cache[i]);
                g_big_cache.erase(g_big_cache.begin() + i);
                return cudaSuccess;
            }
    }
    cudaError_t e = cudaMalloc(out, bytes);
    if (e == cudaErrorMemoryAllocation) {       // buffers of other sizes may be sitting idle in the caches: give them back, once
        cudaGetLastError();
        if (release_caches() > 0) e = cudaMalloc(out, bytes);
    }
    if (e == cudaSuccess && bytes >= (1u << 20)) {
        std::lock_guard<std::mutex> lock(g_big_mutex);
        g_big_live.push_back({*out, bytes, device});
    }
    return e;
}
template <typename T> cudaError_t big_malloc(T **out, size_t bytes) { return big_malloc_impl(reinterpret_cast<void **>(out), bytes); }

void big_free(void *p)
{
    if (!p) return;
    {
        std::lock_guard<std::mutex> lock(g_big_mutex);
        for (size_t i = 0; i < g_big_live.size(); ++i)
            if (g_big_live[i].ptr == p) {
                const BigBuffer b = g_big_live[i];
                g_big_live.erase(g_big_live.begin() + i);
                size_t total = b.bytes;
                for (const BigBuffer &c : g_big_cache) total += c.bytes;
                if (total <= big_cache_limit()) { g_big_cache.push_back(b); return; }
                break;
            }
    }
    cudaFree(p);
}
constexpr size_t kQueueEntryBytes = 3 * 16 + 4;    // three uint4 arrays and one float array (SlabParams)

int fail(int code, const std::string &msg)
{
    g_last_error = msg;
    return code;
}

#define SOC_CUDA(call)                                                                              \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess)                                                                      \
            return fail(SOC_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));             \
    } while (0)

constexpr double kPi = 3.14159265358979323846;
constexpr double kWMin = 1e-9;          // termination threshold relative to the initial weight (reading S7)
constexpr int kChunk = 64;              // package ids a warp claims from the global counter at a time
constexpr unsigned kFull = 0xffffffffu;

// Bounds-checked build (-DSOC_CHECKED; paper_1812_06632_b200/build.py --checked -> libsoc_b200_checked.so): every index
// into a global or shared array of the photon kernels is tested against the array's length; a violation is counted
// (soc_checked_violations) and the access redirected to element 0.  The stand-in for compute-sanitizer memcheck on
// boxes where the sanitizer cannot run; compiled out of the product library.
#ifdef SOC_CHECKED
__device__ unsigned int g_violations = 0;
__device__ __forceinline__ long long ck_index(long long i, long long n)
{
    if (i < 0 || i >= n) { atomicAdd(&g_violations, 1u); return 0; }
    return i;
}
#define CK(i, n) ck_index((long long)(i), (long long)(n))
#else
#define CK(i, n) (i)
#endif

struct DevResult {                      // one slot per launch, accumulated with atomics
    double emitted, escaped, absorbed;
    unsigned long long cell_steps, scatterings, terminated;
    unsigned int drift_bits, pad_;      // fp32 bits of max |w - (1 - sum of deposits)| over the packages that escaped
    unsigned long long gathers, reds;   // option "stats": global-memory gather / reduction instructions issued by the lanes
    unsigned long long suspensions, refusals;   // slab-blocked launches: states queued by the walk / refused by a full queue
};

// f1: dust re-emission, the third package source.  Package ids [n_const, n_const + n_dust)
struct DustParams {
    long long n_const, n_dust;          // ids below n_const are background / point-source packages
    unsigned long long stride;          // id -> (id * stride) mod n_dust spreads consecutive ids over the cells
    const uint32_t *first;              // [n_total + 1] first dust index of every cell (prefix sums of count)
    const int32_t *count;               // [n_total] packages per cell
    const float *T;                     // [n_total] dust temperature
    double *self_abs;                   // [n_total] or NULL: in-cell absorption of the cells' own packages (f3)
    double kabs, freq_hz, weight;       // luminosity L_c = 4 pi kabs rho h^3 B_nu(T); weight of the self_abs adds
    int n_levels;
    int level_off[SOC_MAX_LEVELS + 1];  // ABI cell vector: first global id of every level
};

struct SimParams {
    // grid
    int nx, ny, nz, n_root;
    int n_total, n_oct;                 // lengths of cellw / parent (bounds-checked build)
    const uint32_t *cellw;              // [n_total] leaf: fp32 density bits; parent: 0x80000000 | (first child id - n_root)
    const int32_t *parent;              // [n_octets] (parent id - n_root) of octet (id - n_root) >> 3
    // dust at this frequency
    double kabs, ksca, g;
    // sources
    int is_beam, n_point;
    long long n_bg;
    double bg_e0, surf;
    double beam[6];
    double ps_pos[SOC_MAX_POINT_SOURCES][3];
    double ps_e0[SOC_MAX_POINT_SOURCES];
    DustParams dust;
    // run
    long long pkg_begin, pkg_end;
    unsigned long long seed;
    int ifreq;
    int refill_threshold;
    double weight;
    double *absorbed;
    soc_replay_record *replay;
    unsigned long long *counter;
    DevResult *result;
};

}  // namespace

struct soc_grid {
    int nx = 0, ny = 0, nz = 0, n_levels = 0, n_freq = 0;
    long long n_total = 0, n_root = 0, n_octets = 0;
    long long level_off[SOC_MAX_LEVELS + 1] = {0};
    std::vector<double> freq, kabs, ksca, g;
    uint32_t *d_cellw = nullptr;
    int32_t *d_parent = nullptr;
    DevResult *d_results = nullptr;           // n_slots
    unsigned long long *d_counters = nullptr; // n_slots
    DevResult *h_results = nullptr;           // pinned, n_slots
    float *d_table = nullptr;
    // f1 / f3: dust re-emission
    uint32_t *d_dust_first = nullptr;         // [n_total + 1] prefix sums of the package counts of the current launch
    uint32_t *d_scan_blocks = nullptr;        // block sums of the scan
    double *d_scalars = nullptr;              // [8] small reductions (sum of luminosities, emitting cells, packages)
    double *h_scalars = nullptr;              // pinned mirror
    double *d_freqtab = nullptr;              // [3][n_freq] freq_hz, kabs, quadrature weight
    double *d_eff = nullptr;                  // [n_total] effective absorbed energy of the ALI update
    float *h_table = nullptr;                 // pinned staging copy of the caller's table (borrowed for the call only)
    cudaEvent_t ev_table = nullptr;           // the staging copy has been read
    // internal layout of the production kernel: root grid with one ghost layer, then the octet levels
    int nbx = 0, nby = 0, nbz = 0, nrp = 0;
    long long n_int = 0;
    uint32_t *d_cellw_int = nullptr;
    int32_t *d_parent_int = nullptr;
    double *d_acc = nullptr;                  // [n_int], zero between calls
    float *d_acc32 = nullptr;                 // [n_int], zero between calls (fp32 internal accumulator)
    // soc_simulate_spectrum overlaps consecutive frequencies on two streams (the tail of one launch, where lanes run
    // out of packages, is filled by the next): a second set of accumulators and the stream / events that order them
    float *d_acc32_b = nullptr;
    double *d_acc_b = nullptr;
    int acc_sel = 0;                          // accumulator set the next launch uses
    int overlap_active = 0, last_overlap = 0, opt_overlap = 1;
    cudaStream_t aux = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr, ev_unpad[2] = {nullptr, nullptr};
    cudaEvent_t unpad_wait = nullptr;         // the next fold into the caller's array waits for this one
    int opt_acc32 = 1;
    int n_slots = 0;
    int device = 0, n_sm = 0;
    long long l2_bytes = 126ll << 20;   // cudaDevAttrL2CacheSize of the grid's device (B200: 126 MB), set by soc_grid_create
    int opt_blocks_per_sm = 0;                // 0 = from the occupancy calculator
    int opt_threads = 256;
    int opt_refill_threshold = 1;
    int opt_service_threshold = 0;            // parked lanes that trigger a service pass; 0 = by scattering depth (8 or 16)
    int opt_hot_cache = 1;
    int opt_stats = 0;                        // production kernels count their gather / reduction instructions (slower variant)
    int opt_carveout = -1;                    // preferred shared-memory carve-out of the photon kernels in %, -1 = driver default
    double rho_mean = 0.0;                    // mean density of the root-level leaves
    int opt_kernel = 0;                       // regular grids: 0 = by working-set size, 1 = photon_fast_kernel, 2 = photon_q_kernel
    // z-slab blocking (SlabParams): package queues of the two accumulator sets
    int opt_slabs = 0;                        // 0 = by working-set size, 1 = off, n >= 2 = n slabs
    int opt_slab_sweeps = 0;                  // sweeps over the slabs before the final whole-grid phase; 0 = 2
    long long opt_slab_queue_limit = 0;       // test hook: entries a queue accepts from the walk; 0 = its capacity
    long long opt_slab_chunk = 0;             // test hook: packages per sequence of phases; 0 = 2^24
    int opt_group = 0;                        // frequencies per launch of soc_simulate_spectrum: 0 = by package count, 1..4
    std::vector<int> slot_group;              // [n_slots] size of the grouped launch that starts at this result slot, else 0
    double *d_hot64[2] = {nullptr, nullptr};  // hot-cell sums of the two accumulator sets (FastParams::hot64)
    uint4 *d_slab_q[2] = {nullptr, nullptr};  // 3 arrays of n_slabs * cap entries
    unsigned *d_slab_cnt[2] = {nullptr, nullptr};
    size_t slab_q_entries[2] = {0, 0};
    int opt_timing = 0;                       // record a CUDA-event pair around every photon launch
    std::vector<cudaEvent_t> ev0, ev1;        // n_slots each (created on demand)
    std::vector<char> ev_set;
    cudaEvent_t ev_after_photon = nullptr;
};

// The working-set thresholds of the kernel choice were measured on B200's 126 MB of L2 (64 MB: photon_q_kernel instead of
// photon_fast_kernel; 96 MB: slab blocking, in slabs of 80 MB); on another device they scale with its L2.
static inline long long l2_share(const soc_grid *G, int mb_of_126) { return G->l2_bytes / 126 * mb_of_126; }

// ------------------------------------------------------------------------------------------------
// device code
// ------------------------------------------------------------------------------------------------
namespace {

// a1: Philox4x32-10 (Salmon et al. 2011), counter (block, pkg_lo, pkg_hi, ifreq), key (seed_lo, seed_hi)
__device__ __forceinline__ void philox_block(unsigned long long seed, int ifreq, long long pkg, uint32_t block,
                                             uint32_t &o0, uint32_t &o1, uint32_t &o2, uint32_t &o3)
{
    uint32_t c0 = block, c1 = (uint32_t)((unsigned long long)pkg), c2 = (uint32_t)((unsigned long long)pkg >> 32),
             c3 = (uint32_t)ifreq;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

// word -> ((x >> 9) + 0.5) 2^-23, exact in fp32 and fp64
template <typename R> __device__ __forceinline__ R uniform01(uint32_t w)
{
    return (R)(2u * (w >> 9) + 1u) * (R)(1.0 / 16777216.0);
}

template <typename R> struct RM;
template <> struct RM<float> {
    static __device__ __forceinline__ float sqrt_(float x) { return sqrtf(x); }
    static __device__ __forceinline__ float log_(float x) { return logf(x); }
    static __device__ __forceinline__ void sincospi_(float x, float *s, float *c) { sincospif(x, s, c); }
    static __device__ __forceinline__ float inf() { return __int_as_float(0x7f800000); }
    static __device__ __forceinline__ float copysign_(float a, float b) { return copysignf(a, b); }
    static __device__ __forceinline__ float rsqrt_(float x) { return rsqrtf(x); }
};
template <> struct RM<double> {
    static __device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
    static __device__ __forceinline__ double log_(double x) { return log(x); }
    static __device__ __forceinline__ void sincospi_(double x, double *s, double *c) { sincospi(x, s, c); }
    static __device__ __forceinline__ double inf() { return __longlong_as_double(0x7ff0000000000000ll); }
    static __device__ __forceinline__ double copysign_(double a, double b) { return copysign(a, b); }
    static __device__ __forceinline__ double rsqrt_(double x) { return 1.0 / sqrt(x); }
};

// Precision (reading S11): the package state (position in the cell, direction, remaining optical
// depth) is fp32; A is the type the updates are evaluated in before they are rounded back to fp32:
//   A = float  : production (SOC_GEOM_FP32)
//   A = double : replay (SOC_GEOM_FP64) -- the same evaluation as the fp64 oracle up to 1e-16, so the
//                rounded fp32 state stays bit-identical except within 2^-29 of a rounding boundary.
template <typename A> __device__ __forceinline__ float clamp01f(A x)
{
    return (float)(x < (A)0 ? (A)0 : (x > (A)1 ? (A)1 : x));
}

// per-lane package state
template <typename A> struct Pkg {
    float fx, fy, fz;      // position inside the cell, units of the cell edge, [0,1]
    float dx, dy, dz;      // direction (unit length up to fp32 rounding)
    A rx, ry, rz;          // 1 / direction, in the arithmetic type
    float tau_rem;         // remaining scattering optical depth of the flight segment
    float h;               // cell edge 2^-(level-1), exact
    int ix, iy, iz;        // root cell
    int rel;               // HIER: cell id - n_root (< 0: root cell, level 1); regular grid: cell id
    uint32_t cw;           // cell word of the current cell (fp32 density bits for a leaf)
    uint32_t w_hg, w_az;   // words 1, 2 of the current segment's Philox block
    uint32_t seg, steps, scat;
    unsigned long long hash;
    double E, e_min;       // weight and termination threshold 1e-9 E0
    double pend;           // energy absorbed in the current cell, not yet added to the accumulator
    long long id;
    int origin;            // dust package that has not left the cell that emitted it: that cell's global id; else -1
};

template <typename A> __device__ __forceinline__ void set_direction(Pkg<A> &p, A dx, A dy, A dz)
{
    p.dx = (float)dx; p.dy = (float)dy; p.dz = (float)dz;
    p.rx = (A)1 / (A)p.dx; p.ry = (A)1 / (A)p.dy; p.rz = (A)1 / (A)p.dz;
}

// a6: descend to the leaf that holds the position; 2f and 2f-1 are exact in fp32
template <typename A> __device__ __forceinline__ void descend(const SimParams &P, Pkg<A> &p)
{
    uint32_t cw = __ldg(P.cellw + CK(p.rel + P.n_root, P.n_total));
    while ((int32_t)cw < 0) {
        int slot = 0;
        if (p.fx >= 0.5f) { slot |= 1; p.fx = 2.0f * p.fx - 1.0f; } else p.fx = 2.0f * p.fx;
        if (p.fy >= 0.5f) { slot |= 2; p.fy = 2.0f * p.fy - 1.0f; } else p.fy = 2.0f * p.fy;
        if (p.fz >= 0.5f) { slot |= 4; p.fz = 2.0f * p.fz - 1.0f; } else p.fz = 2.0f * p.fz;
        p.rel = (int)(cw & 0x7fffffffu) + slot;
        p.h *= 0.5f;
        cw = __ldg(P.cellw + CK(p.rel + P.n_root, P.n_total));
    }
    p.cw = cw;
}

// f1: luminosity of leaf cell at (level, rho, T): L = 4 pi kabs rho h^3 B_nu(T), in the energy unit of pi I S
__device__ __forceinline__ double planck_nu(double nu, double T)
{
    if (!(T > 0.0)) return 0.0;
    const double h = 6.62607015e-27, kb = 1.380649e-16, c = 2.99792458e10;
    return 2.0 * h * nu * nu * nu / (c * c) / expm1(h * nu / (kb * T));
}

__device__ __forceinline__ double cell_luminosity(double kabs, double freq_hz, uint32_t cw, int level0, float T)
{
    if ((int32_t)cw < 0) return 0.0;                                // parent cell
    const double rho = (double)__uint_as_float(cw);
    if (!(rho > 0.0)) return 0.0;
    const double vol = 1.0 / (double)(1ull << (3 * level0));         // level0 = level - 1
    return 4.0 * 3.14159265358979323846 * kabs * rho * vol * planck_nu(freq_hz, (double)T);
}

// f1: the cell that emits dust package `id` (global id of the ABI cell vector) and its level - 1
__device__ __forceinline__ int dust_cell(const DustParams &D, long long id, int &level0)
{
    const unsigned long long q = ((unsigned long long)(id - D.n_const) * D.stride) % (unsigned long long)D.n_dust;
    int lo = 0, hi = D.level_off[D.n_levels];                       // invariant: first[lo] <= q < first[hi]
    while (hi - lo > 1) {
        const int mid = (int)(((long long)lo + hi) >> 1);
        if ((unsigned long long)__ldg(D.first + CK(mid, D.level_off[D.n_levels] + 1)) <= q) lo = mid; else hi = mid;
    }
    level0 = 0;
    while (level0 + 1 < D.n_levels && lo >= D.level_off[level0 + 1]) ++level0;
    return lo;
}

// a1-a3: position, root cell, direction and source of package `id` (SURVEY.md 8c.3 / DESIGN.md readings S2, S3).
// One definition for both kernels families: A = double in the replay kernel, float in the production kernels; PARAMS
// is SimParams or FastParams (same field names).  src = point source index, -1 = background or beam.
// Dust packages (f1): src = -2, ix = global id of the emitting cell, iy = its level - 1; uniform point in the cell,
// isotropic direction (words 0..2 of block 0 -> position, word 3 -> cos theta, word 0 of block 1 -> azimuth).
template <typename A, typename PARAMS>
__device__ __forceinline__ void emit_core(const PARAMS &P, int ifreq, long long id, int &ix, int &iy, int &iz, float &fx, float &fy,
                                          float &fz, A &dx, A &dy, A &dz, int &src)
{
    src = -1;
    if (!P.is_beam && id >= P.dust.n_const) {
        uint32_t w0, w1, w2, w3, v0, v1, v2, v3;
        philox_block(P.seed, ifreq, id, 0u, w0, w1, w2, w3);
        philox_block(P.seed, ifreq, id, 1u, v0, v1, v2, v3);
        ix = dust_cell(P.dust, id, iy);
        iz = 0;
        fx = uniform01<float>(w0); fy = uniform01<float>(w1); fz = uniform01<float>(w2);       // exact in fp32
        const A mu = (A)2 * uniform01<A>(w3) - (A)1;
        const A st = RM<A>::sqrt_(fmax((A)0, fma(-mu, mu, (A)1)));
        A sp, cp;
        RM<A>::sincospi_((A)2 * uniform01<A>(v0), &sp, &cp);
        dx = st * cp; dy = st * sp; dz = mu;
        src = -2;
        return;
    }
    if (P.is_beam) {
        const int n[3] = {P.nx, P.ny, P.nz};
        int c[3];
        float f[3];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            int i = (int)floor(P.beam[j]);
            i = i > n[j] - 1 ? n[j] - 1 : i;
            c[j] = i;
            f[j] = (float)(P.beam[j] - (double)i);
        }
        ix = c[0]; iy = c[1]; iz = c[2];
        fx = f[0]; fy = f[1]; fz = f[2];
        dx = (A)P.beam[3]; dy = (A)P.beam[4]; dz = (A)P.beam[5];
    } else if (id < P.n_bg) {
        uint32_t w0, w1, w2, w3, v0, v1, v2, v3;
        philox_block(P.seed, ifreq, id, 0u, w0, w1, w2, w3);
        philox_block(P.seed, ifreq, id, 1u, v0, v1, v2, v3);
        // face in proportion to its area, order x-, x+, y-, y+, z-, z+ (exact in fp64 like the definition)
        const double ax = (double)P.ny * P.nz, ay = (double)P.nz * P.nx, az = (double)P.nx * P.ny;
        const double x = uniform01<double>(w0) * P.surf;
        int face = 5;
        if (x < ax) face = 0;
        else if (x < 2 * ax) face = 1;
        else if (x < 2 * ax + ay) face = 2;
        else if (x < 2 * ax + 2 * ay) face = 3;
        else if (x < 2 * ax + 2 * ay + az) face = 4;
        const int a = face >> 1, high = face & 1;
        const int n1 = a == 0 ? P.ny : (a == 1 ? P.nz : P.nx);     // extent along a1 = (a+1)%3
        const int n2 = a == 0 ? P.nz : (a == 1 ? P.nx : P.ny);     // extent along a2 = (a+2)%3
        const int na = a == 0 ? P.nx : (a == 1 ? P.ny : P.nz);
        // u*N = (2k+1) N / 2^24: integer cell and fraction, rounded once to fp32 like fl32(u*N - i)
        const unsigned long long m1 = (unsigned long long)(2u * (w1 >> 9) + 1u) * (unsigned)n1;
        const unsigned long long m2 = (unsigned long long)(2u * (w2 >> 9) + 1u) * (unsigned)n2;
        const int i1 = (int)(m1 >> 24), i2 = (int)(m2 >> 24);
        const float f1 = (float)(uint32_t)(m1 & 0xffffffu) * (float)(1.0 / 16777216.0);
        const float f2 = (float)(uint32_t)(m2 & 0xffffffu) * (float)(1.0 / 16777216.0);
        const int ia = high ? na - 1 : 0;
        const float fa = high ? 1.0f : 0.0f;
        const A u3 = uniform01<A>(w3);
        const A mu = RM<A>::sqrt_(u3), st = RM<A>::sqrt_((A)1 - u3);
        A sp, cp;
        RM<A>::sincospi_((A)2 * uniform01<A>(v0), &sp, &cp);
        const A da = high ? -mu : mu, d1 = st * cp, d2 = st * sp;
        if (a == 0)      { ix = ia; iy = i1; iz = i2; fx = fa; fy = f1; fz = f2; dx = da; dy = d1; dz = d2; }
        else if (a == 1) { iy = ia; iz = i1; ix = i2; fy = fa; fz = f1; fx = f2; dy = da; dz = d1; dx = d2; }
        else             { iz = ia; ix = i1; iy = i2; fz = fa; fx = f1; fy = f2; dz = da; dx = d1; dy = d2; }
    } else {
        uint32_t w0, w1, w2, w3;
        philox_block(P.seed, ifreq, id, 0u, w0, w1, w2, w3);
        const int k = (int)((id - P.n_bg) % P.n_point);
        const double px = P.ps_pos[k][0], py = P.ps_pos[k][1], pz = P.ps_pos[k][2];
        ix = (int)floor(px); iy = (int)floor(py); iz = (int)floor(pz);
        fx = (float)(px - (double)ix); fy = (float)(py - (double)iy); fz = (float)(pz - (double)iz);
        const A mu = fma((A)2, uniform01<A>(w0), (A)-1);
        const A st = RM<A>::sqrt_(fmax((A)0, fma(-mu, mu, (A)1)));
        A sp, cp;
        RM<A>::sincospi_((A)2 * uniform01<A>(w1), &sp, &cp);
        dx = st * cp; dy = st * sp; dz = mu;
        src = k;
    }
}

// a8: new direction after a scattering: Henyey-Greenstein polar angle in the cancellation-free form (reading S6) from
// word w_hg, azimuth from word w_az, rotation in the basis of Duff et al. 2017 (reading in SURVEY.md 8c.7), renormalised.
template <typename A>
__device__ __forceinline__ void scatter_direction(A g, uint32_t w_hg, uint32_t w_az, A odx, A ody, A odz, A &ndx, A &ndy, A &ndz)
{
    // every a * b + c below is written as an explicit fma: the two production kernels inline this function in different
    // surroundings, and must not be left to contract it differently (they are tested to walk identical paths)
    const A mu0 = fma((A)2, uniform01<A>(w_hg), (A)-1);
    const A m2 = mu0 * mu0, g2 = g * g;
    const A num = fma(g2 * g, (m2 - (A)1) * (A)0.5, fma(g2, mu0, fma(g, ((A)3 + m2) * (A)0.5, mu0)));
    const A gm = fma(g, mu0, (A)1);
    A ct = num / (gm * gm);
    ct = ct > (A)1 ? (A)1 : (ct < (A)-1 ? (A)-1 : ct);
    const A st = RM<A>::sqrt_(fmax((A)0, fma(-ct, ct, (A)1)));
    A sp, cp;
    RM<A>::sincospi_((A)2 * uniform01<A>(w_az), &sp, &cp);
    const A sg = RM<A>::copysign_((A)1, odz);
    const A a = (A)-1 / (sg + odz);
    const A b = odx * ody * a;
    const A t1x = fma(sg * odx, odx * a, (A)1), t1y = sg * b, t1z = -sg * odx;
    const A t2x = b, t2y = fma(ody, ody * a, sg), t2z = -ody;
    const A c1 = st * cp, c2 = st * sp;
    const A nx = fma(c1, t1x, fma(c2, t2x, ct * odx));
    const A ny = fma(c1, t1y, fma(c2, t2y, ct * ody));
    const A nz = fma(c1, t1z, fma(c2, t2z, ct * odz));
    const A inv = RM<A>::rsqrt_(fma(nx, nx, fma(ny, ny, nz * nz)));
    ndx = nx * inv; ndy = ny * inv; ndz = nz * inv;
}

// a1-a4: create package `id` in the replay kernel's state
template <typename A, bool HIER>
__device__ __forceinline__ double emit(const SimParams &P, Pkg<A> &p, long long id)
{
    A dx, dy, dz;
    int src;
    p.id = id;
    emit_core<A>(P, P.ifreq, id, p.ix, p.iy, p.iz, p.fx, p.fy, p.fz, dx, dy, dz, src);
    double e0 = P.is_beam ? 1.0 : (src >= 0 ? P.ps_e0[src] : P.bg_e0);
    set_direction(p, dx, dy, dz);
    p.h = 1.0f;
    p.origin = -1;
    if (src == -2) {
        // f1: the package starts inside the leaf that emitted it; its root cell is found by climbing the reverse links
        const int gid = p.ix, level0 = p.iy;
        p.origin = gid;
        p.cw = __ldg(P.cellw + CK(gid, P.n_total));
        e0 = cell_luminosity(P.dust.kabs, P.dust.freq_hz, p.cw, level0, __ldg(P.dust.T + CK(gid, P.n_total))) /
             (double)__ldg(P.dust.count + CK(gid, P.n_total));
        p.h = __int_as_float((127 - level0) << 23);              // 2^-(level - 1), exact
        int r = HIER ? gid - P.n_root : gid;
        p.rel = r;
        if (HIER) while (r >= 0) r = __ldg(P.parent + CK(r >> 3, P.n_oct));
        const int root = HIER ? r + P.n_root : r;
        p.ix = root % P.nx; p.iy = (root / P.nx) % P.ny; p.iz = root / (P.nx * P.ny);
    } else {
        const int root = p.ix + P.nx * (p.iy + P.ny * p.iz);
        if (HIER) {
            p.rel = root - P.n_root;
            descend(P, p);
        } else {
            p.rel = root;
            p.cw = __ldg(P.cellw + CK(root, P.n_total));
        }
    }
    p.seg = 0; p.steps = 0; p.scat = 0;
    p.hash = 0xcbf29ce484222325ull;
    p.E = e0;
    p.e_min = kWMin * e0;
    p.pend = 0.0;
    uint32_t s0, s1, s2, s3;
    philox_block(P.seed, P.ifreq, id, 2u, s0, s1, s2, s3);
    p.tau_rem = (float)(-RM<A>::log_(uniform01<A>(s0)));          // a4
    p.w_hg = s1; p.w_az = s2;
    return e0;
}

// a8 in the replay kernel: evaluated in A from the fp32 state, rounded once
template <typename A> __device__ __forceinline__ void scatter(const SimParams &P, Pkg<A> &p)
{
    A nx, ny, nz;
    scatter_direction<A>((A)P.g, p.w_hg, p.w_az, (A)p.dx, (A)p.dy, (A)p.dz, nx, ny, nz);
    set_direction(p, nx, ny, nz);
    p.seg += 1; p.scat += 1;
    uint32_t s0, s1, s2, s3;
    philox_block(P.seed, P.ifreq, p.id, 2u + p.seg, s0, s1, s2, s3);
    p.tau_rem = (float)(-RM<A>::log_(uniform01<A>(s0)));
    p.w_hg = s1; p.w_az = s2;
}

// a5/a6: move across the face of axis a in direction sg.  Returns false when the package leaves the grid.
template <typename A, bool HIER>
__device__ __forceinline__ bool move_across(const SimParams &P, Pkg<A> &p, int a, int sg)
{
    if (HIER) {
        // sibling flip, else up to the common parent; (f + bit)/2 rounds once to fp32
        while (p.rel >= 0) {
            const int bit = (p.rel >> a) & 1;
            if ((sg > 0) != (bit != 0)) { p.rel ^= (1 << a); goto found; }
            p.fx = (p.fx + (float)(p.rel & 1)) * 0.5f;
            p.fy = (p.fy + (float)((p.rel >> 1) & 1)) * 0.5f;
            p.fz = (p.fz + (float)((p.rel >> 2) & 1)) * 0.5f;
            p.rel = __ldg(P.parent + CK(p.rel >> 3, P.n_oct));
            p.h *= 2.0f;
        }
    }
    {
        bool out;
        if (a == 0)      { p.ix += sg; out = (unsigned)p.ix >= (unsigned)P.nx; }
        else if (a == 1) { p.iy += sg; out = (unsigned)p.iy >= (unsigned)P.ny; }
        else             { p.iz += sg; out = (unsigned)p.iz >= (unsigned)P.nz; }
        if (out) return false;
        const int root = p.ix + P.nx * (p.iy + P.ny * p.iz);
        p.rel = HIER ? root - P.n_root : root;
    }
found:
    {
        const float face = sg > 0 ? 0.0f : 1.0f;      // entry face in the neighbour's frame
        if (a == 0) p.fx = face; else if (a == 1) p.fy = face; else p.fz = face;
    }
    if (HIER) descend(P, p);
    else p.cw = __ldg(P.cellw + CK(p.rel, P.n_total));
    return true;
}

template <typename A, bool HIER, bool REPLAY>
__global__ void __launch_bounds__(256) photon_kernel(const __grid_constant__ SimParams P)
{
    const int lane = threadIdx.x & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    double acc_emit = 0.0, acc_esc = 0.0, acc_abs = 0.0;
    unsigned long long acc_steps = 0;
    unsigned acc_scat = 0, acc_term = 0;
    Pkg<A> p;
    bool active = false;
    long long pool_next = 0, pool_end = 0;       // warp-uniform id pool
    bool exhausted = false;
    const A ksca = (A)P.ksca;
    const float kabs_f = (float)P.kabs;

    for (;;) {
        unsigned idle = __ballot_sync(kFull, !active);
        if (idle && !exhausted && (__popc(idle) >= P.refill_threshold || idle == kFull)) {
            do {
                if (pool_next >= pool_end) {
                    long long base = 0;
                    if (lane == 0) base = (long long)atomicAdd(P.counter, (unsigned long long)kChunk);
                    base = __shfl_sync(kFull, base, 0) + P.pkg_begin;
                    if (base >= P.pkg_end) { exhausted = true; break; }
                    pool_next = base;
                    pool_end = base + kChunk < P.pkg_end ? base + kChunk : P.pkg_end;
                }
                const long long avail = pool_end - pool_next;
                const int rank = __popc(idle & lt_mask);
                if (!active && rank < avail) {
                    acc_emit += emit<A, HIER>(P, p, pool_next + rank);
                    active = true;
                }
                const int n_idle = __popc(idle);
                pool_next += n_idle < avail ? n_idle : avail;
                idle = __ballot_sync(kFull, !active);
            } while (idle);
        }
        if (idle == kFull) break;                // nothing left for this warp

        if (active) {
            // ---- geometry: distance (in cell edges) to the face of each axis
            const A inf = RM<A>::inf();
            const A tx = p.dx == 0.0f ? inf : ((p.dx > 0.0f ? (A)1 : (A)0) - (A)p.fx) * p.rx;
            const A ty = p.dy == 0.0f ? inf : ((p.dy > 0.0f ? (A)1 : (A)0) - (A)p.fy) * p.ry;
            const A tz = p.dz == 0.0f ? inf : ((p.dz > 0.0f ? (A)1 : (A)0) - (A)p.fz) * p.rz;
            int a = 0;
            A ts = tx;
            if (ty < ts) { a = 1; ts = ty; }         // lowest axis wins a tie (reading S4)
            if (tz < ts) { a = 2; ts = tz; }
            const float rho = __uint_as_float(p.cw);
            const A ds = HIER ? ts * (A)p.h : ts;
            const A ksr = (A)rho * ksca;
            const A dtau = ds * ksr;
            const bool sc = ksr > (A)0 && dtau >= (A)p.tau_rem;
            A ds_u = ds, t_u = ts;
            if (sc) {
                ds_u = (A)p.tau_rem / ksr;
                t_u = HIER ? ds_u / (A)p.h : ds_u;
            }
            // ---- a7: path-length estimator, continuous absorption
            const int gid = HIER ? p.rel + P.n_root : p.rel;
            const float x = (float)ds_u * rho * kabs_f;
            double frac;
            if (x > 4.0f) frac = -expm1(-((double)ds_u * (double)rho * P.kabs));   // rare: keep the tail of the weight
            else frac = (double)(-expm1f(-x));
            double dep = p.E * frac;
            double e_new = p.E - dep;
            const bool term = e_new < p.e_min;      // a9: residual stays in the cell
            if (term) { dep = p.E; e_new = 0.0; }
            p.pend += dep;
            acc_abs += dep;
            p.E = e_new;
            p.steps += 1;
            if (REPLAY) p.hash = (p.hash ^ (unsigned long long)gid) * 0x100000001b3ull;
            bool done = term;
            bool flush = term;
            double e_esc = 0.0;
            if (term) {
                acc_term += 1;
            } else {
                p.fx = clamp01f<A>((A)p.fx + t_u * (A)p.dx);
                p.fy = clamp01f<A>((A)p.fy + t_u * (A)p.dy);
                p.fz = clamp01f<A>((A)p.fz + t_u * (A)p.dz);
                if (sc) {
                    scatter(P, p);
                } else {
                    flush = true;                    // leaving the cell: hand its energy to the accumulator
                    p.tau_rem = (float)((A)p.tau_rem - dtau);
                    const float da = a == 0 ? p.dx : (a == 1 ? p.dy : p.dz);
                    if (!move_across<A, HIER>(P, p, a, da > 0.0f ? 1 : -1)) {
                        e_esc = p.E;
                        acc_esc += p.E;
                        done = true;
                    }
                }
            }
            // scatterings inside one cell are summed in a register: one atomic per cell visit, not per
            // step (the hot-cell contention of PAPER.md:151, 279)
            if (flush) {
                if (p.pend > 0.0) atomicAdd(P.absorbed + CK(gid, P.n_total), P.weight * p.pend);
                if (p.origin >= 0) {                 // f3: what a cell's own package left in it before first leaving it
                    if (P.dust.self_abs && p.pend > 0.0) atomicAdd(P.dust.self_abs + CK(gid, P.n_total), P.weight * p.pend);
                    p.origin = -1;
                }
                p.pend = 0.0;
            }
            if (done) {
                acc_steps += p.steps;
                acc_scat += p.scat;
                if (REPLAY) {
                    soc_replay_record r;
                    r.hash = p.hash; r.steps = p.steps; r.scatters = p.scat; r.e_escaped = e_esc;
                    P.replay[CK(p.id - P.pkg_begin, P.pkg_end - P.pkg_begin)] = r;
                }
                active = false;
            }
        }
    }

    // ---- per-launch totals: warp shuffle reduction, one set of atomics per warp
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        acc_emit += __shfl_xor_sync(kFull, acc_emit, o);
        acc_esc += __shfl_xor_sync(kFull, acc_esc, o);
        acc_abs += __shfl_xor_sync(kFull, acc_abs, o);
        acc_steps += __shfl_xor_sync(kFull, acc_steps, o);
        acc_scat += __shfl_xor_sync(kFull, acc_scat, o);
        acc_term += __shfl_xor_sync(kFull, acc_term, o);
    }
    if (lane == 0 && acc_steps != 0) {
        atomicAdd(&P.result->emitted, acc_emit);
        atomicAdd(&P.result->escaped, acc_esc);
        atomicAdd(&P.result->absorbed, acc_abs);
        atomicAdd(&P.result->cell_steps, acc_steps);
        atomicAdd(&P.result->scatterings, (unsigned long long)acc_scat);
        atomicAdd(&P.result->terminated, (unsigned long long)acc_term);
    }
}


// ------------------------------------------------------------------------------------------------
// production kernel (SOC_GEOM_FP32)
//
// Same method, arranged for the machine:
//   * internal cell layout: the root grid, surrounded by ghost cells, is stored as 2x2x2 bricks of 8
//     consecutive cells (slot = bx + 2 by + 4 bz, exactly like an octet of the hierarchy), so that a brick of
//     fp32 cell words is one 32-byte sector.  Half of all face crossings stay inside the brick (`id ^= 1 << a`,
//     the same sector: an L1 hit instead of an L2 request), the other half add a brick stride.  Leaving the
//     grid is "the loaded cell word is the sentinel": no coordinates are carried and no bounds are tested.
//     The accumulator lives in the same layout and is folded into the caller's array by unpad_add_kernel
//   * the rare, long code (new package: 2-3 Philox blocks + emission; scattering: HG + rotation + Philox +
//     log + 3 reciprocals) is NOT executed where it arises: the lane parks, and the warp services all parked
//     lanes together once `service_threshold` of them wait (or nothing else can run), so that code runs with
//     many lanes active instead of one or two
//   * package weight is carried relative to the initial energy in fp32 (w in [1e-9, 1]); every deposit is
//     w - w_new, so emitted = absorbed + escaped holds per package to fp32 rounding (~1e-7, unbiased), and the
//     scatter-add is (double)(sum of deposits in the cell visit) * E0 into the fp64 accumulator
// ------------------------------------------------------------------------------------------------
constexpr uint32_t kSentinel = 0xffffffffu;       // cell word of a ghost cell

enum : int { RUN = 0, SCAT = 1, DONE = 2, EMPTY = 3, NEWID = 4, DEAD = 5, SUSP = 6 };

// z-slab blocking of regular grids whose working set exceeds L2.  The bricks of the padded root grid are
// stored z-major, so a slab of brick layers is one contiguous id range of the cell words and of the accumulator.  A
// frequency is a sequence of launches ("phases"), each of which serves one slab: it pops that slab's queue, walks the
// packages while they stay inside their slab and SUSPENDS a package that crosses into the next slab -- its state (48
// bytes) goes to that slab's queue and the walk resumes when the slab's turn comes.  The phases sweep the slabs up and
// down; a last phase pops every queue and confines nothing.
//   * A launch pops the entries [head, frozen) of a queue; `frozen` is the tail as it stood when the previous launch
//     ended (written by that launch's last block), so entries pushed while a queue is being popped wait for its next turn
//     and no slot is ever read before it is written.
//   * No tail: a warp that finds its queue empty does not wait for its running lanes -- it DUMPS them (state to a
//     "leftover" queue, popped first by the next phase) and exits, so a phase ends within one service pass of the moment
//     its queue runs dry.  Two leftover queues alternate between consecutive phases.
//   * A queue that is full refuses the package, which then walks on unconfined (sl = -1) in the launch that holds it.
constexpr int kMaxSlabs = 62;          // + 2 leftover queues = 64 queues
constexpr int kSlabChunk = 16;         // queue slots a warp claims at a time
struct SlabParams {
    uint4 *qa, *qb, *qc;                // all queues, queue q from slab_qbase(q): (fx, fy, fz, tau_rem), (dx, dy, dz, w),
                                        // (absrel, idx | class << 25, rel, scat); class = 0 background or beam, 1 + k point
                                        // source k, 126 / 127 dust package that has left / not yet left the cell that sent it
    float *qp;                          // launches with dust packages (f1): energy of the package / e_ref
    unsigned *cnt;                      // [64][4]: head, tail, frozen, entries written by slab_emit_kernel; then the count of
                                        // finished blocks
    unsigned cap, cap_left;             // entries per slab queue / per leftover queue
    unsigned limit, limit_left;         // entries a queue accepts before it refuses a package (= cap, cap_left; less: test hook)
    int n_slabs, slab_ids;              // ids per slab = brick layers per slab * 8 nbx nby
    int q_left;                         // the leftover queue this launch pops (n_slabs or n_slabs + 1); it dumps to the other
    int s_first, s_last;                // slab queues this launch pops, in this order
    int final_phase;                    // nothing is suspended or dumped
    unsigned long long q_entries;       // entries of each of qa, qb, qc, qp (the bounds-checked build tests against it)
};
constexpr int kSlabCntLen = 4 * 64 + 4;                     // elements of SlabParams::cnt
constexpr int kHot64Len = SOC_MAX_POINT_SOURCES * 343;      // elements of FastParams::hot64
__device__ __forceinline__ size_t slab_qbase(const SlabParams &S, int q)
{
    return q < S.n_slabs ? (size_t)q * S.cap : (size_t)S.n_slabs * S.cap + (size_t)(q - S.n_slabs) * S.cap_left;
}
// the last block of a launch to finish: the popped queues were drained up to `frozen`; every queue's new `frozen` is its
// tail now (all pushes of this launch are complete)
__device__ __forceinline__ void slab_epilogue(const SlabParams &S, bool pops)
{
    __shared__ unsigned s_is_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        s_is_last = atomicAdd(S.cnt + CK(4 * 64, kSlabCntLen), 1u) == gridDim.x - 1 ? 1u : 0u;
    }
    __syncthreads();
    if (s_is_last && (int)threadIdx.x < S.n_slabs + 2) {
        const int q = threadIdx.x;
        volatile unsigned *c = S.cnt + CK(4 * q, kSlabCntLen - 3);
        if (pops && (q == S.q_left || (q >= S.s_first && q <= S.s_last))) c[0] = c[2];
        const unsigned t = c[1];
        if (!pops) c[3] = t;                     // slab_emit_kernel: its entries are all in (it never fills a queue)
        unsigned cap = q < S.n_slabs ? S.limit : S.limit_left;
        cap = cap > c[3] ? cap : c[3];
        c[1] = c[2] = t < cap ? t : cap;
        if (q == 0) S.cnt[4 * 64] = 0u;
    }
}

// Grouped launch: a launch of fewer than ~4e6 packages ends with its blocks waiting for their last
// long-lived packages (0.4 ms on B200, a quarter of an octree launch of 1e6 packages), so up to kMaxJobs consecutive
// frequencies share one launch: package g of the launch belongs to job g / job_pkgs, and everything that differs between
// the frequencies is read per lane from this table.  The jobs add into ONE accumulator in units of e_ref, each with its
// quadrature weight folded into its package energies (rel = weight * energy / e_ref).
constexpr int kMaxJobs = 4;
#ifndef SOC_GROUP_MIN_REL
#define SOC_GROUP_MIN_REL 1e-7f
#endif
constexpr float kGroupMinRel = SOC_GROUP_MIN_REL;   // a job's brightest source class, in units of the launch's (enqueue_group)
struct JobParams {
    float ksca, kabs, kratio, g;
    float bg_rel, beam_rel;
    int ifreq, pad_;
    double bg_e0;
    double ps_e0[SOC_MAX_POINT_SOURCES];
    float ps_rel[SOC_MAX_POINT_SOURCES];
};

struct FastParams {
    int nx, ny, nz;                     // root grid
    int nbx, nby;                       // bricks along x, y of the padded root grid (cell ix sits at X = ix + 2)
    int bsy, bsz;                       // id strides between bricks along y, z (along x: 8): 8 nbx, 8 nbx nby
    int nrp;                            // number of padded root cells = 8 nbx nby nbz
    int n_root;                         // nx*ny*nz
    int n_int, n_oct, n_abi, n_replay;  // lengths of cellw / parent / the ABI cell vector / replay (bounds-checked build)
    const uint32_t *cellw;              // [n_int] leaf: fp32 density bits; parent: 0x80000000 | internal id of first child
    const int32_t *parent;              // [n_octets] internal id of the parent of octet (id - nrp) >> 3
    float kabs, ksca, kratio, g;        // kratio = kabs / ksca
    int is_beam, n_point;
    long long n_bg;
    double bg_e0, surf;
    double beam[6];
    double ps_pos[SOC_MAX_POINT_SOURCES][3];
    double ps_e0[SOC_MAX_POINT_SOURCES];
    long long pkg_begin, pkg_end;
    unsigned long long seed;
    int ifreq;
    int service_threshold;
    int hot_r;                          // half-width R of the cached cube around every point source, -1 = no cache
    double *acc;                        // [n_int] internal accumulator (unweighted energies), ACC32 = false
    float *acc32;                       // [n_int] internal accumulator in units of e_ref, ACC32 = true
    double *hot64;                      // [n_point][(2 hot_r + 1)^3] ACC32: the blocks' hot-cell partial sums, in units of e_ref.
                                        // fp64: a cell next to a source collects ~1e5 partial sums per launch, and an fp32
                                        // sum that large silently drops the small ones
    float bg_rel, beam_rel;             // package energy / e_ref of a background / beam package
    float ps_rel[SOC_MAX_POINT_SOURCES];  // ... of a package of point source k
    DustParams dust;
    double e_ref;                       // reference energy of the launch (unit of the fp32 accumulator)
    soc_replay_record *replay;
    unsigned long long *counter;
    DevResult *result;
    SlabParams slab;
    int n_jobs;                         // GROUP launches: jobs of the launch; result + j is the slot of job j
    long long job_pkgs;                 // packages per job: ids [pkg_begin, pkg_begin + job_pkgs) of each frequency
    JobParams job[kMaxJobs];
};

struct FPkg {
    float fx, fy, fz;       // position inside the cell, [0,1]
    float dx, dy, dz;       // direction
    float rx, ry, rz;       // 1/d (+-inf where d == 0)
    float tau_rem, h;
    float w, pend, absrel;  // weight / E0; deposits of this cell visit; deposits of this package
    int rel;                // internal cell id
    uint32_t cw;
    uint32_t steps, scat;   // scat is also the index of the current flight segment
    int src;                // point source index, -1 = background or beam
    int anc1, anc2, anc3;   // hierarchy: ids of the parent, grandparent and great-grandparent of the current cell (the
                            // package's own path down, shifted on every descent / climb; -1 = not known), so that
                            // climbing to the common parent loads no reverse links for the last three levels descended
    int disp;               // hot-cell tracking: packed (dx + R) | (dy + R) << 8 | (dz + R) << 16 relative to the
                            // source cell while the package is inside the cached cube, else -1
    long long id;
    unsigned long long hash;
    uint32_t n_ld, n_red;   // REPLAY variants only (option "stats"): gathers / reductions issued for this package
    uint32_t w_hg, w_az;    // regular grids: words 1, 2 of the current segment's Philox block (the scattering that ends the
                            // segment takes its angles from them: kept, so that the block is computed once)
    int job;                // GROUP launches: the frequency of the launch this package belongs to
};

// Distance to the exit face along axis a, in cell edges:  t_a = (d_a > 0 ? 1 - f_a : -f_a) / d_a
//   = fma(-f_a, r_a, max(r_a, 0)).   d_a == 0 gives r_a = +-inf and t_a = +inf or NaN; fminf skips a NaN and the
// equality test that picks the axis is false for it, so such an axis is never crossed (as in the definition).
__device__ __forceinline__ float exit_time(float f, float r) { return fmaf(-f, r, fmaxf(r, 0.0f)); }

__device__ __forceinline__ void fast_set_direction(FPkg &p, float dx, float dy, float dz)
{
    p.dx = dx; p.dy = dy; p.dz = dz;
    p.rx = 1.0f / dx; p.ry = 1.0f / dy; p.rz = 1.0f / dz;
}

__device__ __forceinline__ double package_e0(const FastParams &P, int src)
{
    return src >= 0 ? P.ps_e0[src] : (P.is_beam ? 1.0 : P.bg_e0);
}

__device__ __forceinline__ float package_rel(const FastParams &P, int src)
{
    return src >= 0 ? P.ps_rel[src] : (P.is_beam ? P.beam_rel : P.bg_rel);
}

// a6: descend to the leaf.  Returns false on the sentinel (outside the root grid).
__device__ __forceinline__ bool fast_descend(const FastParams &P, FPkg &p)
{
    uint32_t cw = __ldg(P.cellw + CK(p.rel, P.n_int));
    p.n_ld += 1;
    if (cw == kSentinel) { p.cw = cw; return false; }
    while ((int32_t)cw < 0) {
        // 2 f and 2 f - 1 are exact in fp32: one fused operation per axis gives the bits of the two-step form
        const bool bx = p.fx >= 0.5f, by = p.fy >= 0.5f, bz = p.fz >= 0.5f;
        p.fx = fmaf(p.fx, 2.0f, bx ? -1.0f : 0.0f);
        p.fy = fmaf(p.fy, 2.0f, by ? -1.0f : 0.0f);
        p.fz = fmaf(p.fz, 2.0f, bz ? -1.0f : 0.0f);
        const int slot = (bx ? 1 : 0) | (by ? 2 : 0) | (bz ? 4 : 0);
        p.anc3 = p.anc2; p.anc2 = p.anc1; p.anc1 = p.rel;       // the cell being left becomes the parent
        p.rel = (int)(cw & 0x7fffffffu) + slot;
        p.h *= 0.5f;
        cw = __ldg(P.cellw + CK(p.rel, P.n_int));
        p.n_ld += 1;
    }
    p.cw = cw;
    return true;
}

// internal id of root cell (ix, iy, iz): brick (X>>1, Y>>1, Z>>1), slot (X&1) + 2 (Y&1) + 4 (Z&1), X = ix + 2
__device__ __forceinline__ int root_id(const FastParams &P, int ix, int iy, int iz)
{
    const int X = ix + 2, Y = iy + 2, Z = iz + 2;
    return 8 * ((X >> 1) + P.nbx * ((Y >> 1) + P.nby * (Z >> 1))) + (X & 1) + 2 * (Y & 1) + 4 * (Z & 1);
}

// global id (ABI cell vector) of an internal id -- only the replay records need it
__device__ __forceinline__ long long global_id(const FastParams &P, int rel)
{
    if (rel >= P.nrp) return (long long)(rel - P.nrp) + P.n_root;
    const int B = rel >> 3, bz = B / (P.nbx * P.nby), r = B - bz * (P.nbx * P.nby), by = r / P.nbx, bx = r - by * P.nbx;
    const int ix = 2 * bx + (rel & 1) - 2, iy = 2 * by + ((rel >> 1) & 1) - 2, iz = 2 * bz + ((rel >> 2) & 1) - 2;
    return ix + (long long)P.nx * (iy + (long long)P.ny * iz);
}

// a1-a3 in the production kernels: the direction is returned, not installed
__device__ __forceinline__ void fast_emit_core(const FastParams &P, FPkg &p, int ifreq, long long id, int &ix, int &iy, int &iz,
                                               float &dx, float &dy, float &dz)
{
    p.id = id;
    emit_core<float>(P, ifreq, id, ix, iy, iz, p.fx, p.fy, p.fz, dx, dy, dz, p.src);
}

// prel receives the package energy in units of the launch's reference energy
template <bool HIER>
__device__ __forceinline__ void fast_emit(const FastParams &P, FPkg &p, int ifreq, long long id, float &dx, float &dy, float &dz, float &prel)
{
    int ix, iy, iz;
    fast_emit_core(P, p, ifreq, id, ix, iy, iz, dx, dy, dz);
    p.h = 1.0f;
    p.n_ld = 0; p.n_red = 0;
    if (HIER) p.anc1 = p.anc2 = p.anc3 = -1;
    if (p.src == -2) {
        // f1: a dust package starts inside the leaf that emitted it (ix = its global id, iy = its level - 1); the ids
        // of its ancestors are not known (-1): a climb loads the reverse links
        const int gid = ix, level0 = iy;
        if (gid < P.n_root) p.rel = root_id(P, gid % P.nx, (gid / P.nx) % P.ny, gid / (P.nx * P.ny));
        else p.rel = P.nrp + (gid - P.n_root);
        p.cw = __ldg(P.cellw + CK(p.rel, P.n_int));
        p.n_ld = 1;
        p.h = __int_as_float((127 - level0) << 23);
        const double e0 = cell_luminosity(P.dust.kabs, P.dust.freq_hz, p.cw, level0, __ldg(P.dust.T + CK(gid, P.n_abi))) /
                          (double)__ldg(P.dust.count + CK(gid, P.n_abi));
        prel = (float)(e0 / P.e_ref);
    } else {
        p.rel = root_id(P, ix, iy, iz);
        if (HIER) fast_descend(P, p);
        else { p.cw = __ldg(P.cellw + CK(p.rel, P.n_int)); p.n_ld = 1; }
        prel = package_rel(P, p.src);
    }
    // hot-cell tracking starts at the centre of the cube of the package's own source (regular grids only)
    p.disp = (!HIER && p.src >= 0 && P.hot_r >= 0) ? P.hot_r * 0x010101 : -1;
    p.steps = 0; p.scat = 0;
    p.hash = 0xcbf29ce484222325ull;
    p.w = 1.0f; p.pend = 0.0f; p.absrel = 0.0f;
}

// a7: new weight w e^-x and deposit w (1 - e^-x) for x >= 0.  Below x = 1/8 the deposit is w times the series
//   x - x^2/2 + x^3/6 - x^4/24 + x^5/120   (relative error < 5e-8)
// and the weight is reduced by it, so that a deposit far below the fp32 resolution of the weight (x ~ 1e-8 per cell at
// millimetre wavelengths) is still added to the cell with full relative accuracy; above, the weight is w e^-x and the
// deposit the difference.
__device__ __forceinline__ void absorb(float w, float x, float &w_new, float &dep)
{
    const float e = expf(-x);
    const float small = x * fmaf(x, fmaf(x, fmaf(x, fmaf(x, 1.0f / 120.0f, -1.0f / 24.0f), 1.0f / 6.0f), -0.5f), 1.0f);
    const bool lo = x < 0.125f;
    const float d_lo = w * small, w_hi = w * e;
    w_new = lo ? w - d_lo : w_hi;
    dep = lo ? d_lo : w - w_hi;
}

// the same, bit for bit, with the exponential behind a warp-uniform branch: at most wavelengths no lane of a warp ever has
// x >= 1/8, and expf is a fifth of the arithmetic of a cell-step
__device__ __forceinline__ void absorb_v(float w, float x, float &w_new, float &dep)
{
    const float small = x * fmaf(x, fmaf(x, fmaf(x, fmaf(x, 1.0f / 120.0f, -1.0f / 24.0f), 1.0f / 6.0f), -0.5f), 1.0f);
    const bool lo = x < 0.125f;
    const float d_lo = w * small;
    w_new = w - d_lo;
    dep = d_lo;
    if (__any_sync(__activemask(), !lo)) {
        const float w_hi = w * expf(-x);
        if (!lo) { w_new = w_hi; dep = w - w_hi; }
    }
}

// a9: weight with which a package leaves the grid, relative to its initial energy.  The sum of the deposits
// (`absrel`) resolves a small absorbed fraction, the running weight a small remainder: take the one that is accurate
// (they differ by accumulated fp32 rounding only)
__device__ __forceinline__ double escaped_rel(float w, float absrel)
{
    if (w == 0.0f) return 0.0;                   // terminated: the residual was deposited
    return absrel < 0.5f ? 1.0 - (double)absrel : (double)w;
}

// DUST: the launch contains dust re-emission packages (f1): per-package energies, in-cell absorption (f3).  Compiled out of
// the kernels that serve the constant sources, whose step loop it would lengthen (measured: -4 % ... -10 %).
// GROUP: the launch carries the packages of several frequencies (JobParams).
template <bool HIER, bool REPLAY, bool ACC32, bool DUST, bool GROUP>
__global__ void __launch_bounds__(256, HIER ? 5 : 4) photon_fast_kernel(const __grid_constant__ FastParams P)
{
    static_assert(!GROUP || (ACC32 && !DUST), "grouped launches: constant sources, fp32 accumulator");
    // GROUP: totals per warp and job (touched when a package starts or ends): emitted, escaped, absorbed; cell-steps,
    // scatterings, terminations; weight drift
    __shared__ double s_jd[GROUP ? 8 : 1][kMaxJobs][3];
    __shared__ unsigned long long s_jn[GROUP ? 8 : 1][kMaxJobs][3];
    __shared__ unsigned s_jdrift[GROUP ? 8 : 1][kMaxJobs];
    const int wid = GROUP ? (threadIdx.x >> 5) : 0;
    if (GROUP && threadIdx.x < 8 * kMaxJobs) {
        const int w = threadIdx.x / kMaxJobs, j = threadIdx.x % kMaxJobs;   // (64 threads at least)
        s_jd[w][j][0] = s_jd[w][j][1] = s_jd[w][j][2] = 0.0;
        s_jn[w][j][0] = s_jn[w][j][1] = s_jn[w][j][2] = 0ull;
        s_jdrift[w][j] = 0u;
    }
    const int lane = threadIdx.x & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    double acc_emit = 0.0, acc_esc = 0.0, acc_abs = 0.0;
    unsigned long long acc_steps = 0;
    unsigned acc_scat = 0, acc_term = 0;
    float acc_drift = 0.0f;                      // max |w - (1 - absrel)|: the running weight against the sum of the deposits
    unsigned long long acc_ld = 0, acc_red = 0;  // REPLAY variants: request counters (option "stats")
    FPkg p;
    p.n_ld = 0; p.n_red = 0;
    p.src = -1; p.disp = -1; p.w = 0.0f; p.absrel = 0.0f; p.steps = 0; p.scat = 0; p.cw = 0; p.rel = 0; p.h = 1.0f;
    p.anc1 = p.anc2 = p.anc3 = -1; p.job = 0;
    int need = EMPTY;
    // hot-cell cache (atomics to the cells around a point source serialise): fp32 partial sums
    // of the deposits (in units of the source's package energy) into the (2R+1)^3 root cells around each source
    extern __shared__ float s_hot[];
    __shared__ float s_prel[256];                // dust packages: package energy / e_ref (one per package, not per class)
    const int hot_side = 2 * P.hot_r + 1;
    const int hot_cells = P.hot_r >= 0 ? hot_side * hot_side * hot_side : 0;
    for (int i = threadIdx.x; i < hot_cells * P.n_point; i += blockDim.x) s_hot[i] = 0.0f;
    __syncthreads();
    long long pool_next = 0, pool_end = 0;       // warp-uniform id pool
    bool exhausted = false;
    const int T = P.service_threshold;

    for (;;) {
        const unsigned m_park = __ballot_sync(kFull, (unsigned)(need - SCAT) <= (unsigned)(EMPTY - SCAT));
        const unsigned m_run = __ballot_sync(kFull, need == RUN);
        if (m_park && (__popc(m_park) >= T || m_run == 0u)) {
            // ---------------------------------------------------------------- service, all parked lanes together
            if (need == DONE) {                  // retire the finished package
                const double e0 = GROUP ? (p.src >= 0 ? P.job[p.job].ps_e0[p.src] : P.job[p.job].bg_e0)
                                        : ((DUST && p.src <= -2) ? (double)s_prel[threadIdx.x] * P.e_ref : package_e0(P, p.src));
                const double esc = escaped_rel(p.w, p.absrel) * e0;
                if (GROUP) {
                    atomicAdd(&s_jd[wid][p.job][1], esc);
                    atomicAdd(&s_jd[wid][p.job][2], (double)p.absrel * e0);
                    atomicAdd(&s_jn[wid][p.job][0], (unsigned long long)p.steps);
                    atomicAdd(&s_jn[wid][p.job][1], (unsigned long long)p.scat);
                    if (p.w == 0.0f) atomicAdd(&s_jn[wid][p.job][2], 1ull);
                    else atomicMax(&s_jdrift[wid][p.job], __float_as_uint(fabsf(p.w - (1.0f - p.absrel))));
                } else {
                    if (p.w != 0.0f) acc_drift = fmaxf(acc_drift, fabsf(p.w - (1.0f - p.absrel)));
                    acc_esc += esc;
                    acc_abs += (double)p.absrel * e0;
                    acc_steps += p.steps;
                    acc_scat += p.scat;
                }
                if (REPLAY) {
                    acc_ld += p.n_ld; acc_red += p.n_red;
                    if (P.replay) {
                        soc_replay_record r;
                        r.hash = p.hash; r.steps = p.steps; r.scatters = p.scat; r.e_escaped = esc;
                        P.replay[CK(p.id - P.pkg_begin, P.n_replay)] = r;
                    }
                }
                need = EMPTY;
            }
            unsigned want = __ballot_sync(kFull, need == EMPTY);
            if (want && !exhausted) {
                do {
                    if (pool_next >= pool_end) {
                        long long base = 0;
                        if (lane == 0) base = (long long)atomicAdd(P.counter, (unsigned long long)kChunk);
                        base = __shfl_sync(kFull, base, 0) + P.pkg_begin;
                        if (base >= P.pkg_end) { exhausted = true; break; }
                        pool_next = base;
                        pool_end = base + kChunk < P.pkg_end ? base + kChunk : P.pkg_end;
                    }
                    const long long avail = pool_end - pool_next;
                    const int rank = __popc(want & lt_mask);
                    if (need == EMPTY && rank < avail) { p.id = pool_next + rank; need = NEWID; }
                    const int n_want = __popc(want);
                    pool_next += n_want < avail ? n_want : avail;
                    want = __ballot_sync(kFull, need == EMPTY);
                } while (want);
            }
            if (need == EMPTY && exhausted) need = DEAD;
            float ndx = 0.0f, ndy = 0.0f, ndz = 1.0f;
            if (need == NEWID) {
                float prel;
                if (GROUP) {                     // id of the launch -> job and package id of that frequency
                    const long long g = p.id - P.pkg_begin;
                    p.job = (int)(g / P.job_pkgs);
                    p.id = P.pkg_begin + (g - (long long)p.job * P.job_pkgs);
                }
                fast_emit<HIER>(P, p, GROUP ? P.job[p.job].ifreq : P.ifreq, p.id, ndx, ndy, ndz, prel);
                if (GROUP) {
                    s_prel[threadIdx.x] = p.src >= 0 ? P.job[p.job].ps_rel[p.src] : P.job[p.job].bg_rel;
                    atomicAdd(&s_jd[wid][p.job][0], p.src >= 0 ? P.job[p.job].ps_e0[p.src] : P.job[p.job].bg_e0);
                } else if (DUST && p.src <= -2) { s_prel[threadIdx.x] = prel; acc_emit += (double)prel * P.e_ref; }
                else acc_emit += package_e0(P, p.src);
            } else if (need == SCAT) {
                // finish the flight segment: advance to the scattering point (a4), then a8
                const float rho = __uint_as_float(p.cw);
                float t_u = p.tau_rem / (rho * (GROUP ? P.job[p.job].ksca : P.ksca));
                if (HIER) t_u /= p.h;
                p.fx = __saturatef(fmaf(t_u, p.dx, p.fx));
                p.fy = __saturatef(fmaf(t_u, p.dy, p.fy));
                p.fz = __saturatef(fmaf(t_u, p.dz, p.fz));
                uint32_t s0, w_hg, w_az, s3;     // words 1, 2 of the block of the segment that ends here
                if (HIER) philox_block(P.seed, GROUP ? P.job[p.job].ifreq : P.ifreq, p.id, 2u + p.scat, s0, w_hg, w_az, s3);
                else { w_hg = p.w_hg; w_az = p.w_az; }
                scatter_direction<float>(GROUP ? P.job[p.job].g : P.g, w_hg, w_az, p.dx, p.dy, p.dz, ndx, ndy, ndz);
                p.scat += 1;
            }
            if (need == NEWID || need == SCAT) {
                fast_set_direction(p, ndx, ndy, ndz);
                uint32_t s0, s1, s2, s3;
                philox_block(P.seed, GROUP ? P.job[p.job].ifreq : P.ifreq, p.id, 2u + p.scat, s0, s1, s2, s3);
                if (!HIER) { p.w_hg = s1; p.w_az = s2; }                      // (the octree kernel has no registers to spare)
                p.tau_rem = -__logf(uniform01<float>(s0));                    // a4
                need = RUN;
                if (HIER && p.cw == kSentinel) need = DONE;                   // cannot happen for valid sources
            }
            continue;
        }
        if (m_run == 0u) break;                  // nothing parked that can be serviced, nothing running

        // four cell-steps per look at the warp's state: the ballots and the loop overhead are paid once; a lane
        // that parks in one of them sits out the rest
        auto cell_step = [&]() {
            // ---------------------------------------------------------------- one cell-step (a5-a7, a9)
            const float rho = __uint_as_float(p.cw);
            const float tx = exit_time(p.fx, p.rx);
            const float ty = exit_time(p.fy, p.ry);
            const float tz = exit_time(p.fz, p.rz);
            const float ts = fminf(fminf(tx, ty), tz);
            const bool ax0 = tx == ts, ax1 = !ax0 && ty == ts;       // lowest axis wins a tie (reading S4)
            const float da = ax0 ? p.dx : (ax1 ? p.dy : p.dz);
            const bool fwd = da > 0.0f;
            const int bstride = ax0 ? 8 : (ax1 ? P.bsy : P.bsz);      // to the same slot of the next brick
            const int abit = ax0 ? 1 : (ax1 ? 2 : 4);
            const float tsh = HIER ? ts * p.h : ts;
            const float ksr = rho * (GROUP ? P.job[p.job].ksca : P.ksca);
            const float dtau = tsh * ksr;
            const bool sc = dtau >= p.tau_rem && ksr > 0.0f;
            const float x = sc ? p.tau_rem * (GROUP ? P.job[p.job].kratio : P.kratio) : tsh * (rho * (GROUP ? P.job[p.job].kabs : P.kabs));
            float w_new, dep;
            if (HIER) absorb_v(p.w, x, w_new, dep);      // (measured: the branch pays on the octree, not on the regular grids)
            else absorb(p.w, x, w_new, dep);
            const bool term = w_new < (float)kWMin;                  // a9: residual stays in the cell
            if (term) { dep = p.w; w_new = 0.0f; }
            p.pend += dep;
            p.absrel += dep;
            p.w = w_new;
            p.steps += 1;
            if (REPLAY)                          // the record hashes cell ids of the ABI's cell vector
                p.hash = (p.hash ^ (unsigned long long)global_id(P, p.rel)) * 0x100000001b3ull;
            if (term || !sc) {
                // the package leaves the cell (or ends in it): hand the cell visit's energy to the accumulator --
                // to the block's shared partial sums while the cell is in the cached cube around the package's
                // source, with one fp64 reduction to L2 otherwise
                if (p.disp >= 0) {
                    const int j = (p.disp & 255) + hot_side * (((p.disp >> 8) & 255) + hot_side * (p.disp >> 16));
                    // (GROUP: already in the launch's unit -- the frequencies of the launch share the partial sums)
                    atomicAdd(s_hot + CK(p.src * hot_cells + j, hot_cells * P.n_point), GROUP ? p.pend * s_prel[threadIdx.x] : p.pend);
                } else if (p.pend > 0.0f) {
                    const bool dust = (DUST && p.src <= -2) || GROUP;    // the package's own unit, kept in shared memory
                    if (ACC32) atomicAdd(P.acc32 + CK(p.rel, P.n_int), p.pend * (dust ? s_prel[threadIdx.x] : package_rel(P, p.src)));
                    else atomicAdd(P.acc + CK(p.rel, P.n_int), (double)p.pend * (dust ? (double)s_prel[threadIdx.x] * P.e_ref : package_e0(P, p.src)));
                    p.n_red += 1;
                }
                if (DUST && p.src == -2) {       // f3: what a cell's own package leaves in it before first leaving it
                    if (P.dust.self_abs && p.pend > 0.0f)
                        atomicAdd(P.dust.self_abs + CK(global_id(P, p.rel), P.n_abi), P.dust.weight * (double)p.pend * ((double)s_prel[threadIdx.x] * P.e_ref));
                    p.src = -3;
                }
                p.pend = 0.0f;
            }
            if (term) {
                if (!GROUP) acc_term += 1;       // (GROUP: counted per job at retirement)
                need = DONE;
            } else if (sc) {
                need = SCAT;                     // the segment is finished in the service block
            } else {
                p.tau_rem -= dtau;
                if (!HIER && p.disp >= 0) {      // follow the package through the cached cube
                    const int sh = ax0 ? 0 : (ax1 ? 8 : 16);
                    const int nd = p.disp + ((fwd ? 1 : -1) << sh);
                    p.disp = ((nd >> sh) & 255) < hot_side ? nd : -1;
                }
                p.fx = __saturatef(fmaf(ts, p.dx, p.fx));
                p.fy = __saturatef(fmaf(ts, p.dy, p.fy));
                p.fz = __saturatef(fmaf(ts, p.dz, p.fz));
                const float face = fwd ? 0.0f : 1.0f;    // entry face in the neighbour's frame
                // neighbour inside the brick / octet: flip the slot bit.  Otherwise, for an octet, go up to the
                // common parent; for a root brick, the same slot bit flips and the brick changes.
                int rel = p.rel;
                bool inside = fwd == ((rel & abit) == 0);
                if (HIER) {
                    while (!inside && rel >= P.nrp) {
                        // (f + b) / 2 = fl(f / 2 + b / 2): halving is exact, so the fused form rounds the same sum once
                        p.fx = fmaf(p.fx, 0.5f, (rel & 1) ? 0.5f : 0.0f);
                        p.fy = fmaf(p.fy, 0.5f, (rel & 2) ? 0.5f : 0.0f);
                        p.fz = fmaf(p.fz, 0.5f, (rel & 4) ? 0.5f : 0.0f);
                        if (p.anc1 >= 0) {
                            rel = p.anc1;
                        } else {                 // the lane does not know this ancestor: reverse link of the octet
                            rel = __ldg(P.parent + CK((rel - P.nrp) >> 3, P.n_oct));
                            p.n_ld += 1;
                        }
                        p.anc1 = p.anc2; p.anc2 = p.anc3; p.anc3 = -1;
                        p.h *= 2.0f;
                        inside = fwd == ((rel & abit) == 0);
                    }
                }
                rel ^= abit;
                if (!inside) rel += fwd ? bstride : -bstride;
                p.rel = rel;
                if (ax0) p.fx = face; else if (ax1) p.fy = face; else p.fz = face;
                if (HIER) {
                    if (!fast_descend(P, p)) need = DONE;            // a9: escaped
                } else {
                    p.cw = __ldg(P.cellw + CK(rel, P.n_int));
                    p.n_ld += 1;
                    if (p.cw == kSentinel) need = DONE;              // a9: escaped
                }
            }
        };
        if (need == RUN) cell_step();
        if (need == RUN) cell_step();
        if (need == RUN) cell_step();
        if (need == RUN) cell_step();
    }

    // ---- the block's hot-cell partial sums go to the accumulator: one fp64 reduction per touched cell and block
    if (hot_cells > 0) {
        __syncthreads();
        for (int i = threadIdx.x; i < hot_cells * P.n_point; i += blockDim.x) {
            const float v = s_hot[i];
            if (v != 0.0f) {
                const int k = i / hot_cells, j = i - k * hot_cells;
                const int jz = j / (hot_side * hot_side), jr = j - jz * hot_side * hot_side, jy = jr / hot_side, jx = jr - jy * hot_side;
                const int ix = (int)floor(P.ps_pos[k][0]) + jx - P.hot_r, iy = (int)floor(P.ps_pos[k][1]) + jy - P.hot_r,
                          iz = (int)floor(P.ps_pos[k][2]) + jz - P.hot_r;
                if (ACC32) atomicAdd(P.hot64 + CK(i, kHot64Len), GROUP ? (double)v : (double)v * (double)P.ps_rel[k]);
                else atomicAdd(P.acc + CK(root_id(P, ix, iy, iz), P.n_int), (double)v * P.ps_e0[k]);
            }
        }
    }

    // ---- per-launch totals: warp shuffle reduction, one set of atomics per warp
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        acc_emit += __shfl_xor_sync(kFull, acc_emit, o);
        acc_esc += __shfl_xor_sync(kFull, acc_esc, o);
        acc_abs += __shfl_xor_sync(kFull, acc_abs, o);
        acc_steps += __shfl_xor_sync(kFull, acc_steps, o);
        acc_scat += __shfl_xor_sync(kFull, acc_scat, o);
        acc_term += __shfl_xor_sync(kFull, acc_term, o);
        acc_drift = fmaxf(acc_drift, __shfl_xor_sync(kFull, acc_drift, o));
    }
    if (GROUP) {
        // per-job totals of this warp -> the result slots of the jobs
        __syncwarp();
        if (lane < P.n_jobs && (s_jn[wid][lane][0] != 0ull || s_jd[wid][lane][0] != 0.0)) {
            DevResult *r = P.result + lane;
            atomicAdd(&r->emitted, s_jd[wid][lane][0]);
            atomicAdd(&r->escaped, s_jd[wid][lane][1]);
            atomicAdd(&r->absorbed, s_jd[wid][lane][2]);
            atomicAdd(&r->cell_steps, s_jn[wid][lane][0]);
            atomicAdd(&r->scatterings, s_jn[wid][lane][1]);
            atomicAdd(&r->terminated, s_jn[wid][lane][2]);
            atomicMax(&r->drift_bits, s_jdrift[wid][lane]);
        }
    }
    if (!GROUP && lane == 0 && acc_steps != 0) {
        atomicAdd(&P.result->emitted, acc_emit);
        atomicAdd(&P.result->escaped, acc_esc);
        atomicAdd(&P.result->absorbed, acc_abs);
        atomicAdd(&P.result->cell_steps, acc_steps);
        atomicAdd(&P.result->scatterings, (unsigned long long)acc_scat);
        atomicAdd(&P.result->terminated, (unsigned long long)acc_term);
        atomicMax(&P.result->drift_bits, __float_as_uint(acc_drift));     // >= 0: fp32 order = integer order
    }
    if (REPLAY) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            acc_ld += __shfl_xor_sync(kFull, acc_ld, o);
            acc_red += __shfl_xor_sync(kFull, acc_red, o);
        }
        if (lane == 0) { atomicAdd(&P.result->gathers, acc_ld); atomicAdd(&P.result->reds, acc_red); }
    }
}

// ------------------------------------------------------------------------------------------------
// production kernel, regular grids: photon_fast_kernel with the lane holding HALF A BRICK in registers
//
// ncu on config 5 (profiles/README.md, round 1): the lane-per-package walk is bound by the number of L1->L2
// requests (tag look-ups 73 % of peak, L1->XBAR request path 67 %), 0.83 gathers + 0.97 scatter-adds per cell-step,
// every one of them to a different sector; without the scatter-adds the same walk runs 1.7 x faster.  The four cells
// of a brick that share bz (slot & 3 = bx + 2 by) are 16 contiguous, aligned bytes.  The lane keeps the four cell
// words of the half it is in (one 16-byte gather when it enters the half) and four deposit sums (one 16-byte
// red.global.add.v4.f32 when it leaves): a crossing along x or y that stays in the brick -- one step in three --
// costs no memory request at all, and the requests per cell-step drop from 1.8 to about 1.3.
// Also here: the per-launch totals live in shared memory (touched only when a package starts or ends), the
// cell-step count is one 32-bit lane counter, the package id a 32-bit offset, source index and hot-cube position
// share a word -- the eight extra registers fit under the 4-CTAs-per-SM cap.
// ------------------------------------------------------------------------------------------------
struct QPkg {
    float fx, fy, fz;       // position inside the cell, [0,1]
    float dx, dy, dz;       // direction
    float rx, ry, rz;       // 1/d
    float tau_rem;
    float w, absrel;        // weight / E0; deposits of this package
    float pend;             // deposits of the current cell visit
    float prel;             // package energy in units of the launch's reference energy (ACC32)
    int rel;                // internal cell id
    uint32_t q0, q1, q2, q3;    // cell words of the half brick rel & ~3
                            // (the deposits into those four cells, not yet in the accumulator, live in shared memory:
                            //  s_acc[slot][thread] -- indexed by the slot, which registers cannot be)
    uint32_t scat;          // scatterings so far = index of the current flight segment
    uint32_t idx;           // package id - pkg_begin
    int sd;                 // < 0: background or beam; else source index << 16 | valid << 9 | hot-cube cell (3 bits per axis)
    uint32_t steps;         // REPLAY only
    unsigned long long hash;
    uint32_t n_ld, n_red;   // REPLAY only (option "stats"): gathers / reductions issued for this package
    int lo;                 // SLAB only: the package is confined to the ids [lo, lo + span) of its z-slab;
    unsigned span;          // not confined: lo = 0, span = 2^32 - 1
};

__device__ __forceinline__ int v_src(int sd) { return sd < 0 ? -1 : (sd >> 16); }

__device__ __forceinline__ uint32_t q_word(const QPkg &p)
{
    const bool lo = (p.rel & 1) != 0, hi = (p.rel & 2) != 0;
    const uint32_t a = lo ? p.q1 : p.q0, b = lo ? p.q3 : p.q2;
    return hi ? b : a;
}

__device__ __forceinline__ void q_load(const FastParams &P, QPkg &p)
{
    const uint4 v = __ldg(reinterpret_cast<const uint4 *>(P.cellw + CK(p.rel & ~3, P.n_int - 3)));
    p.q0 = v.x; p.q1 = v.y; p.q2 = v.z; p.q3 = v.w;
    p.n_ld += 1;
}

// hand the deposits of the half brick (already in units of the launch's reference energy) to the accumulator:
// one 16-byte reduction
__device__ __forceinline__ void q_flush(const FastParams &P, QPkg &p, float (*s_acc)[256])
{
    const float a0 = s_acc[0][threadIdx.x], a1 = s_acc[1][threadIdx.x], a2 = s_acc[2][threadIdx.x], a3 = s_acc[3][threadIdx.x];
    // nothing to add: empty cells, or the cells around a point source, whose deposits went to the block's shared
    // partial sums -- a reduction of zeros there would bring back the very contention those sums avoid
    if ((a0 + a1) + (a2 + a3) == 0.0f) return;
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(P.acc32 + CK(p.rel & ~3, P.n_int - 3)), "f"(a0), "f"(a1),
                 "f"(a2), "f"(a3) : "memory");
    s_acc[0][threadIdx.x] = 0.0f; s_acc[1][threadIdx.x] = 0.0f; s_acc[2][threadIdx.x] = 0.0f; s_acc[3][threadIdx.x] = 0.0f;
    p.n_red += 1;
}

// SLAB: the launch is one phase of a slab-blocked frequency (SlabParams): packages come from the queues instead of the id
// counter (they were created by slab_emit_kernel), a package that crosses out of its slab's id range is suspended, and a
// warp whose queue has run dry hands its running packages to the next phase.  64 registers at 4 CTAs per SM: at 48 the
// compiler re-materialised the shared-memory addresses of the step (+45 instructions per cell-step), and with the working
// set in L2 the fifth CTA is worth less than that.
template <bool REPLAY, bool DUST, bool SLAB>
__global__ void __launch_bounds__(256, SLAB ? 4 : 5) photon_q_kernel(const __grid_constant__ FastParams P)
{
    const int lane = threadIdx.x & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    // per-launch totals of this thread (touched only in the service block)
    __shared__ double s_tot[3][256];             // emitted, escaped, absorbed
    __shared__ unsigned s_cnt[2][256];           // scatterings, terminated
    __shared__ float s_drift[256];               // max |w - (1 - absrel)| over this thread's escaped packages
    __shared__ float s_acc[4][256];              // this thread's deposits into the four cells of its half brick
    s_drift[threadIdx.x] = 0.0f;
    s_acc[0][threadIdx.x] = 0.0f; s_acc[1][threadIdx.x] = 0.0f; s_acc[2][threadIdx.x] = 0.0f; s_acc[3][threadIdx.x] = 0.0f;
    s_tot[0][threadIdx.x] = 0.0; s_tot[1][threadIdx.x] = 0.0; s_tot[2][threadIdx.x] = 0.0;
    s_cnt[0][threadIdx.x] = 0u; s_cnt[1][threadIdx.x] = 0u;
    extern __shared__ float s_hot[];             // hot-cell partial sums, see photon_fast_kernel
    const int hot_side = 2 * P.hot_r + 1;
    const int hot_cells = P.hot_r >= 0 ? hot_side * hot_side * hot_side : 0;
    for (int i = threadIdx.x; i < hot_cells * P.n_point; i += blockDim.x) s_hot[i] = 0.0f;
    __syncthreads();

    unsigned long long acc_ld = 0, acc_red = 0;  // REPLAY variant: request counters (option "stats")
    QPkg p;
    p.n_ld = 0; p.n_red = 0;
    p.sd = -1; p.w = 0.0f; p.absrel = 0.0f; p.scat = 0; p.rel = 0; p.idx = 0; p.steps = 0; p.hash = 0; p.lo = 0; p.span = 0xffffffffu;
    p.q0 = p.q1 = p.q2 = p.q3 = 0u; p.pend = 0.0f; p.prel = 0.0f;
    p.fx = p.fy = p.fz = 0.5f; p.dx = p.dy = 0.0f; p.dz = 1.0f; p.rx = p.ry = p.rz = 1.0f; p.tau_rem = 0.0f;
    int need = EMPTY;
    unsigned n_steps = 0;                        // cell-steps of this lane (all its packages)
    unsigned n_susp = 0, n_refused = 0;          // SLAB: states this lane queued / packages a full queue refused
    unsigned pool_next = 0, pool_end = 0;        // warp-uniform pool of package offsets (SLAB: of queue slots)
    int cur_q = SLAB ? P.slab.s_first - 1 : 0;   // SLAB: position in the list of queues to pop (s_first - 1 = the leftover queue)
    int pool_q = 0;                              // SLAB: the queue the pool was claimed from
    bool exhausted = false;
    int n_dead = 0;                              // warp-uniform: lanes that will get no more packages
    const unsigned n_pkg = (unsigned)(P.pkg_end - P.pkg_begin);      // the launcher keeps this below 2^32
    const int T = P.service_threshold;

    // SLAB: the lanes with `sel` hand their package to queue `dest` (one slot reservation per warp and queue) and become
    // EMPTY; a full queue refuses the package, which then walks on, not confined to a slab any more
    auto push = [&](bool sel, int dest) {
        unsigned todo = __ballot_sync(kFull, sel);
        while (todo) {
            const int leader = __ffs(todo) - 1;
            const int d = __shfl_sync(kFull, dest, leader);
            const bool mine = sel && dest == d;
            const unsigned m = __ballot_sync(kFull, mine);
            unsigned b = 0;
            if (lane == leader) b = atomicAdd(P.slab.cnt + CK(4 * d + 1, kSlabCntLen), (unsigned)__popc(m));
            b = __shfl_sync(kFull, b, leader);
            if (mine) {
                const unsigned slot = b + __popc(m & lt_mask);
                unsigned room = d < P.slab.n_slabs ? P.slab.limit : P.slab.limit_left;
                if (slot >= room) { const unsigned emitted = P.slab.cnt[CK(4 * d + 3, kSlabCntLen)]; room = room > emitted ? room : emitted; }
                if (slot < room) {
                    const size_t e = CK(slab_qbase(P.slab, d) + slot, P.slab.q_entries);
                    const uint32_t cls = (DUST && p.sd <= -2) ? (uint32_t)(129 + p.sd) : (uint32_t)(v_src(p.sd) + 1);
                    const uint32_t tag = p.idx | (cls << 25);
                    if (DUST) P.slab.qp[e] = p.prel;
                    P.slab.qa[e] = make_uint4(__float_as_uint(p.fx), __float_as_uint(p.fy), __float_as_uint(p.fz), __float_as_uint(p.tau_rem));
                    P.slab.qb[e] = make_uint4(__float_as_uint(p.dx), __float_as_uint(p.dy), __float_as_uint(p.dz), __float_as_uint(p.w));
                    P.slab.qc[e] = make_uint4(__float_as_uint(p.absrel), tag, (uint32_t)p.rel, p.scat);
                    if (REPLAY) { acc_ld += p.n_ld; acc_red += p.n_red + 3; }        // + the three 16-byte stores of the state
                    n_susp += 1;
                    need = EMPTY;
                } else {
                    n_refused += 1;
                    p.lo = 0; p.span = 0xffffffffu;
                    q_load(P, p);
                    need = RUN;
                }
            }
            todo &= ~m;
        }
    };

    for (;;) {
        const unsigned m_run = __ballot_sync(kFull, need == RUN);
        const int n_park = 32 - __popc(m_run) - n_dead;
        if (n_park > 0 && (n_park >= T || m_run == 0u)) {
            // ---------------------------------------------------------------- service, all parked lanes together
            if (SLAB) push(need == SUSP, p.lo / P.slab.slab_ids + (p.rel >= p.lo + P.slab.slab_ids ? 1 : -1));
            if (need == DONE) {                  // retire the finished package
                q_flush(P, p, s_acc);
                const int src = v_src(p.sd);
                const double e0 = (DUST && p.sd <= -2) ? (double)p.prel * P.e_ref : package_e0(P, src);
                const double esc = escaped_rel(p.w, p.absrel) * e0;
                if (p.w != 0.0f) s_drift[threadIdx.x] = fmaxf(s_drift[threadIdx.x], fabsf(p.w - (1.0f - p.absrel)));
                s_tot[1][threadIdx.x] += esc;
                s_tot[2][threadIdx.x] += (double)p.absrel * e0;
                s_cnt[0][threadIdx.x] += p.scat;
                if (p.w == 0.0f) s_cnt[1][threadIdx.x] += 1u;            // terminated (a package that escapes has w >= 1e-9)
                if (REPLAY) {
                    acc_ld += p.n_ld; acc_red += p.n_red;
                    if (P.replay) {
                        soc_replay_record r;
                        r.hash = p.hash; r.steps = p.steps; r.scatters = p.scat; r.e_escaped = esc;
                        P.replay[CK(p.idx, P.n_replay)] = r;
                    }
                }
                need = EMPTY;
            }
            unsigned want = __ballot_sync(kFull, need == EMPTY);
            if (want && !exhausted) {
                do {
                    if (SLAB) {
                        // entries [head, frozen) of the leftover queue, then of the slab queues
                        while (pool_next >= pool_end && cur_q <= P.slab.s_last) {
                            const int q = cur_q < P.slab.s_first ? P.slab.q_left : cur_q;
                            const unsigned frozen = P.slab.cnt[CK(4 * q + 2, kSlabCntLen)];
                            unsigned base = 0;
                            if (lane == 0) base = atomicAdd(P.slab.cnt + CK(4 * q, kSlabCntLen), (unsigned)kSlabChunk);
                            base = __shfl_sync(kFull, base, 0);
                            if (base >= frozen) { cur_q += 1; continue; }
                            pool_next = base;
                            pool_end = frozen - base > (unsigned)kSlabChunk ? base + kSlabChunk : frozen;
                            pool_q = q;
                        }
                        if (pool_next >= pool_end) { exhausted = true; break; }
                    } else if (pool_next >= pool_end) {
                        unsigned long long base = 0;
                        if (lane == 0) base = atomicAdd(P.counter, (unsigned long long)kChunk);
                        base = __shfl_sync(kFull, base, 0);
                        if (base >= (unsigned long long)n_pkg) { exhausted = true; break; }
                        pool_next = (unsigned)base;
                        pool_end = n_pkg - pool_next > (unsigned)kChunk ? pool_next + kChunk : n_pkg;
                    }
                    const unsigned avail = pool_end - pool_next;
                    const unsigned rank = __popc(want & lt_mask);
                    if (need == EMPTY && rank < avail) { p.idx = pool_next + rank; p.sd = SLAB ? pool_q : p.sd; need = NEWID; }
                    const unsigned n_want = __popc(want);
                    pool_next += n_want < avail ? n_want : avail;
                    want = __ballot_sync(kFull, need == EMPTY);
                } while (want);
            }
            if (!SLAB) {
                if (need == EMPTY && exhausted) need = DEAD;
                n_dead = __popc(__ballot_sync(kFull, need == DEAD));
            }
            float ndx = 0.0f, ndy = 0.0f, ndz = 1.0f;
            if (SLAB && need == NEWID) {
                // resume a package: slot p.idx of queue p.sd (reciprocals and the half brick are not part of the state)
                const size_t e = CK(slab_qbase(P.slab, p.sd) + p.idx, P.slab.q_entries);
                const uint4 a = P.slab.qa[e], b = P.slab.qb[e], c = P.slab.qc[e];
                p.fx = __uint_as_float(a.x); p.fy = __uint_as_float(a.y); p.fz = __uint_as_float(a.z); p.tau_rem = __uint_as_float(a.w);
                p.dx = __uint_as_float(b.x); p.dy = __uint_as_float(b.y); p.dz = __uint_as_float(b.z); p.w = __uint_as_float(b.w);
                p.rx = 1.0f / p.dx; p.ry = 1.0f / p.dy; p.rz = 1.0f / p.dz;
                p.absrel = __uint_as_float(c.x); p.rel = (int)c.z; p.scat = c.w;
                p.idx = c.y & 0xffffffu;
                const int src = (int)(c.y >> 25) - 1;
                p.sd = -1;
                if (DUST && src >= 125) {        // a dust package: -3 = has left its cell, -2 = not yet (f3 counts what it leaves there)
                    p.sd = src - 128;
                } else if (src >= 0) {
                    // hot-cube tracking (deposits near the package's own source go to the block's partial sums) is not part
                    // of the queued state: the position in the cube follows from the cell
                    p.sd = src << 16;
                    if (P.hot_r >= 0) {
                        const int B = p.rel >> 3, bz = B / (P.nbx * P.nby), r = B - bz * (P.nbx * P.nby), by = r / P.nbx, bx = r - by * P.nbx;
                        const int hx = 2 * bx + (p.rel & 1) - 2 - (int)floor(P.ps_pos[src][0]) + P.hot_r;
                        const int hy = 2 * by + ((p.rel >> 1) & 1) - 2 - (int)floor(P.ps_pos[src][1]) + P.hot_r;
                        const int hz = 2 * bz + ((p.rel >> 2) & 1) - 2 - (int)floor(P.ps_pos[src][2]) + P.hot_r;
                        if ((unsigned)hx < (unsigned)hot_side && (unsigned)hy < (unsigned)hot_side && (unsigned)hz < (unsigned)hot_side)
                            p.sd |= 0x200 | hx | (hy << 3) | (hz << 6);
                    }
                }
                p.prel = (DUST && p.sd <= -2) ? P.slab.qp[e] : package_rel(P, src);
                p.pend = 0.0f;
                p.n_ld = 3; p.n_red = 0;         // ("stats": the three 16-byte loads of the state count as gathers)
                p.lo = 0; p.span = 0xffffffffu;
                if (!P.slab.final_phase) {
                    const int sl = p.rel / P.slab.slab_ids;
                    p.lo = (sl < P.slab.n_slabs ? sl : P.slab.n_slabs - 1) * P.slab.slab_ids;
                    p.span = (unsigned)P.slab.slab_ids;
                }
                q_load(P, p);
                need = RUN;
            } else if (!SLAB && need == NEWID) {
                FPkg q;
                fast_emit<false>(P, q, P.ifreq, P.pkg_begin + (long long)p.idx, ndx, ndy, ndz, p.prel);
                p.fx = q.fx; p.fy = q.fy; p.fz = q.fz; p.rel = q.rel;
                p.n_ld = 0;
                q_load(P, p);
                p.sd = q.src < 0 ? q.src : ((q.src << 16) | (P.hot_r >= 0 ? (0x200 | (P.hot_r * 0x49)) : 0));   // -1 / -2 (dust)
                p.w = 1.0f; p.absrel = 0.0f; p.scat = 0; p.pend = 0.0f;
                p.steps = 0; p.hash = 0xcbf29ce484222325ull;
                p.n_red = 0;                      // (n_ld = 1: the q_load above)
                s_tot[0][threadIdx.x] += (DUST && q.src <= -2) ? (double)p.prel * P.e_ref : package_e0(P, q.src);
            } else if (need == SCAT) {
                // finish the flight segment: advance to the scattering point (a4), then a8
                const float rho = __uint_as_float(q_word(p));
                const float t_u = p.tau_rem / (rho * P.ksca);
                p.fx = __saturatef(fmaf(t_u, p.dx, p.fx));
                p.fy = __saturatef(fmaf(t_u, p.dy, p.fy));
                p.fz = __saturatef(fmaf(t_u, p.dz, p.fz));
                uint32_t s0, w_hg, w_az, s3;     // words 1, 2 of the block of the segment that ends here
                philox_block(P.seed, P.ifreq, P.pkg_begin + (long long)p.idx, 2u + p.scat, s0, w_hg, w_az, s3);
                scatter_direction<float>(P.g, w_hg, w_az, p.dx, p.dy, p.dz, ndx, ndy, ndz);
                p.scat += 1;
            }
            if (need == NEWID || need == SCAT) {
                p.dx = ndx; p.dy = ndy; p.dz = ndz;
                p.rx = 1.0f / ndx; p.ry = 1.0f / ndy; p.rz = 1.0f / ndz;
                uint32_t s0, s1, s2, s3;
                philox_block(P.seed, P.ifreq, P.pkg_begin + (long long)p.idx, 2u + p.scat, s0, s1, s2, s3);
                p.tau_rem = -__logf(uniform01<float>(s0));                    // a4
                need = RUN;
            }
            if (SLAB && exhausted && !P.slab.final_phase) {
                // the queue has run dry: the phase ends here for this warp.  Its running packages (those still confined to
                // a slab) are handed to the next phase in mid-cell: deposits so far to the sums, sums to the accumulator
                const bool dump = need == RUN && p.span != 0xffffffffu;
                if (dump) {
                    if (p.sd >= 0 && (p.sd & 0x200)) {
                        const int j = (p.sd & 7) + hot_side * (((p.sd >> 3) & 7) + hot_side * ((p.sd >> 6) & 7));
                        atomicAdd(s_hot + CK((p.sd >> 16) * hot_cells + j, hot_cells * P.n_point), p.pend);
                    } else {
                        s_acc[CK(p.rel & 3, 4)][CK(threadIdx.x, 256)] += p.pend * p.prel;
                    }
                    if (DUST && p.sd == -2 && P.dust.self_abs && p.pend > 0.0f)      // f3: the part left in its own cell so far
                        atomicAdd(P.dust.self_abs + CK(global_id(P, p.rel), P.n_abi), P.dust.weight * (double)p.pend * ((double)p.prel * P.e_ref));
                    p.pend = 0.0f;
                    q_flush(P, p, s_acc);
                }
                push(dump, P.slab.q_left ^ P.slab.n_slabs ^ (P.slab.n_slabs + 1));
            }
            if (SLAB) {
                if (need == EMPTY && exhausted) need = DEAD;
                n_dead = __popc(__ballot_sync(kFull, need == DEAD));
            }
            continue;
        }
        if (m_run == 0u) break;                  // nothing parked that can be serviced, nothing running

        // four cell-steps per look at the warp's state: the ballots and the loop overhead are paid once; a lane
        // that parks in one of them sits out the rest
        auto cell_step = [&]() {
            // ---------------------------------------------------------------- one cell-step (a5-a7, a9)
            // the geometry of the step does not need the cell word: it goes first, so that the gather issued by the last
            // crossing has that much longer to arrive
            const float tx = exit_time(p.fx, p.rx);
            const float ty = exit_time(p.fy, p.ry);
            const float tz = exit_time(p.fz, p.rz);
            const float ts = fminf(fminf(tx, ty), tz);
            const bool ax0 = tx == ts, ax1 = !ax0 && ty == ts;           // lowest axis wins a tie (reading S4)
            const float da = ax0 ? p.dx : (ax1 ? p.dy : p.dz);
            const bool fwd = da > 0.0f;
            const int bstride = ax0 ? 8 : (ax1 ? P.bsy : P.bsz);          // to the same slot of the next brick (selected
                                                                          // here, not where it is used: measured)
            const int abit = ax0 ? 1 : (ax1 ? 2 : 4);
            const float gx = __saturatef(fmaf(ts, p.dx, p.fx));           // position after a crossing
            const float gy = __saturatef(fmaf(ts, p.dy, p.fy));
            const float gz = __saturatef(fmaf(ts, p.dz, p.fz));
            const uint32_t cw = q_word(p);
            if (cw == kSentinel) {
                need = DONE;                     // a9: the cell entered by the last crossing is outside the grid
            } else {
                const float rho = __uint_as_float(cw);
                const float ksr = rho * P.ksca;
                const float dtau = ts * ksr;
                const bool sc = dtau >= p.tau_rem && ksr > 0.0f;
                const float x = sc ? p.tau_rem * P.kratio : ts * (rho * P.kabs);
                float w_new, dep;
                absorb_v(p.w, x, w_new, dep);
                const bool term = w_new < (float)kWMin;                  // a9: residual stays in the cell
                if (term) { dep = p.w; w_new = 0.0f; }
                p.pend += dep;
                p.absrel += dep;
                p.w = w_new;
                n_steps += 1;
                if (REPLAY) {                    // the record hashes cell ids of the ABI's cell vector
                    p.steps += 1;
                    p.hash = (p.hash ^ (unsigned long long)global_id(P, p.rel)) * 0x100000001b3ull;
                }
                const bool hot = p.sd >= 0 && (p.sd & 0x200);
                if (term || !sc) {
                    // the package leaves the cell (or ends in it): the cell visit's energy goes to the half-brick sums --
                    // inside the cached cube around the package's source to the block's shared partial sums
                    //
                    if (hot) {
                        const int j = (p.sd & 7) + hot_side * (((p.sd >> 3) & 7) + hot_side * ((p.sd >> 6) & 7));
                        atomicAdd(s_hot + CK((p.sd >> 16) * hot_cells + j, hot_cells * P.n_point), p.pend);
                    } else {
                        s_acc[CK(p.rel & 3, 4)][CK(threadIdx.x, 256)] += p.pend * p.prel;
                    }
                    if (DUST && p.sd == -2) {    // f3: what a cell's own package leaves in it before first leaving it
                        if (P.dust.self_abs && p.pend > 0.0f)
                            atomicAdd(P.dust.self_abs + CK(global_id(P, p.rel), P.n_abi), P.dust.weight * (double)p.pend * ((double)p.prel * P.e_ref));
                        p.sd = -3;
                    }
                    p.pend = 0.0f;
                }
                if (term) {
                    need = DONE;                 // the service block flushes the half-brick sums and counts the termination
                } else if (sc) {
                    need = SCAT;                 // the segment is finished in the service block
                } else {
                    p.tau_rem -= dtau;
                    if (hot) {                   // follow the package through the cached cube
                        const int sh = ax0 ? 0 : (ax1 ? 3 : 6);
                        const int c = ((p.sd >> sh) & 7) + (fwd ? 1 : -1);
                        if ((unsigned)c < (unsigned)hot_side) p.sd = (p.sd & ~(7 << sh)) | (c << sh);
                        else p.sd &= ~0x200;
                    }
                    p.fx = gx; p.fy = gy; p.fz = gz;
                    const float face = fwd ? 0.0f : 1.0f;    // entry face in the neighbour's frame
                    if (ax0) p.fx = face; else if (ax1) p.fy = face; else p.fz = face;
                    // neighbour inside the brick: flip the slot bit; otherwise the same bit flips and the brick changes
                    const bool inside = fwd == ((p.rel & abit) == 0);
                    if (!inside || abit == 4) {
                        q_flush(P, p, s_acc);    // leaving the half brick: its sums go out, the new half comes in
                        int rel = p.rel ^ abit;
                        if (!inside) rel += fwd ? bstride : -bstride;
                        p.rel = rel;
                        if (SLAB && (unsigned)(rel - p.lo) >= p.span) need = SUSP;      // into the next slab
                        else q_load(P, p);
                    } else {
                        p.rel ^= abit;
                    }
                }
            }
        };
        if (need == RUN) cell_step();
        if (need == RUN) cell_step();
        if (need == RUN) cell_step();
        if (need == RUN) cell_step();
    }

    // ---- the block's hot-cell partial sums go to the accumulator: one reduction per touched cell and block
    if (hot_cells > 0) {
        __syncthreads();
        for (int i = threadIdx.x; i < hot_cells * P.n_point; i += blockDim.x) {
            const float v = s_hot[i];
            if (v != 0.0f) {
                atomicAdd(P.hot64 + CK(i, kHot64Len), (double)v * (double)P.ps_rel[i / hot_cells]);
            }
        }
    }

    // ---- per-launch totals: warp shuffle reduction, one set of atomics per warp
    double acc_emit = s_tot[0][threadIdx.x], acc_esc = s_tot[1][threadIdx.x], acc_abs = s_tot[2][threadIdx.x];
    unsigned long long acc_steps = n_steps;
    unsigned acc_scat = s_cnt[0][threadIdx.x], acc_term = s_cnt[1][threadIdx.x];
    float acc_drift = s_drift[threadIdx.x];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        acc_emit += __shfl_xor_sync(kFull, acc_emit, o);
        acc_esc += __shfl_xor_sync(kFull, acc_esc, o);
        acc_abs += __shfl_xor_sync(kFull, acc_abs, o);
        acc_steps += __shfl_xor_sync(kFull, acc_steps, o);
        acc_scat += __shfl_xor_sync(kFull, acc_scat, o);
        acc_term += __shfl_xor_sync(kFull, acc_term, o);
        acc_drift = fmaxf(acc_drift, __shfl_xor_sync(kFull, acc_drift, o));
    }
    if (lane == 0 && (acc_steps != 0 || acc_emit != 0.0)) {
        atomicMax(&P.result->drift_bits, __float_as_uint(acc_drift));
    }
    if (REPLAY) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            acc_ld += __shfl_xor_sync(kFull, acc_ld, o);
            acc_red += __shfl_xor_sync(kFull, acc_red, o);
        }
        if (lane == 0) { atomicAdd(&P.result->gathers, acc_ld); atomicAdd(&P.result->reds, acc_red); }
    }
    if (lane == 0 && (acc_steps != 0 || acc_emit != 0.0)) {
        atomicAdd(&P.result->emitted, acc_emit);
        atomicAdd(&P.result->escaped, acc_esc);
        atomicAdd(&P.result->absorbed, acc_abs);
        atomicAdd(&P.result->cell_steps, acc_steps);
        atomicAdd(&P.result->scatterings, (unsigned long long)acc_scat);
        atomicAdd(&P.result->terminated, (unsigned long long)acc_term);
    }
    if (SLAB) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            n_susp += __shfl_xor_sync(kFull, n_susp, o);
            n_refused += __shfl_xor_sync(kFull, n_refused, o);
        }
        if (lane == 0 && n_susp) atomicAdd(&P.result->suspensions, (unsigned long long)n_susp);
        if (lane == 0 && n_refused) atomicAdd(&P.result->refusals, (unsigned long long)n_refused);
        slab_epilogue(P.slab, true);
    }
}

// a1-a4 for a slab-blocked launch: creates every package of the launch (position, direction, first free path) and puts
// it into the queue of the z-slab it starts in.  One package per thread; a block counts its packages per slab in shared
// memory and reserves the slots of a batch of 256 with one atomic per slab.
__global__ void __launch_bounds__(256) slab_emit_kernel(const __grid_constant__ FastParams P)
{
    __shared__ unsigned s_n[kMaxSlabs], s_base[kMaxSlabs];
    const int lane = threadIdx.x & 31;
    const unsigned n_pkg = (unsigned)(P.pkg_end - P.pkg_begin);
    double acc_emit = 0.0;
    for (unsigned base = blockIdx.x * 256u; base < n_pkg; base += gridDim.x * 256u) {      // block-uniform trip count
        if (threadIdx.x < kMaxSlabs) s_n[threadIdx.x] = 0u;
        __syncthreads();
        const unsigned idx = base + threadIdx.x;
        const bool live = idx < n_pkg;
        FPkg q;
        float dx = 0.0f, dy = 0.0f, dz = 1.0f, tau = 0.0f, prel = 0.0f;
        int slab = 0, rel = 0;
        unsigned rank = 0;
        if (live) {
            int ix, iy, iz;
            const long long id = P.pkg_begin + (long long)idx;
            fast_emit_core(P, q, P.ifreq, id, ix, iy, iz, dx, dy, dz);
            if (q.src == -2) {
                // f1: a dust package starts in the cell that sends it (ix = its global id; regular grid); its energy is the
                // cell's luminosity over its package count, in units of the launch's reference energy
                const int gid = ix;
                rel = root_id(P, gid % P.nx, (gid / P.nx) % P.ny, gid / (P.nx * P.ny));
                const double e0 = cell_luminosity(P.dust.kabs, P.dust.freq_hz, __ldg(P.cellw + CK(rel, P.n_int)), 0,
                                                  __ldg(P.dust.T + CK(gid, P.n_abi))) / (double)__ldg(P.dust.count + CK(gid, P.n_abi));
                prel = (float)(e0 / P.e_ref);
                acc_emit += (double)prel * P.e_ref;
            } else {
                rel = root_id(P, ix, iy, iz);
                acc_emit += package_e0(P, q.src);
            }
            uint32_t s0, s1, s2, s3;
            philox_block(P.seed, P.ifreq, id, 2u, s0, s1, s2, s3);
            tau = -__logf(uniform01<float>(s0));                              // a4
            slab = rel / P.slab.slab_ids;
            slab = slab < P.slab.n_slabs ? slab : P.slab.n_slabs - 1;
            rank = atomicAdd(s_n + slab, 1u);
        }
        __syncthreads();
        if ((int)threadIdx.x < P.slab.n_slabs && s_n[threadIdx.x] > 0u)
            s_base[threadIdx.x] = atomicAdd(P.slab.cnt + CK(4 * threadIdx.x + 1, kSlabCntLen), s_n[threadIdx.x]);
        __syncthreads();
        if (live) {
            const size_t e = CK(slab_qbase(P.slab, slab) + CK(s_base[slab] + rank, P.slab.cap), P.slab.q_entries);
            const uint32_t tag = idx | ((q.src == -2 ? 127u : (uint32_t)(q.src + 1)) << 25);
            if (q.src == -2) P.slab.qp[e] = prel;
            P.slab.qa[e] = make_uint4(__float_as_uint(q.fx), __float_as_uint(q.fy), __float_as_uint(q.fz), __float_as_uint(tau));
            P.slab.qb[e] = make_uint4(__float_as_uint(dx), __float_as_uint(dy), __float_as_uint(dz), __float_as_uint(1.0f));
            P.slab.qc[e] = make_uint4(0u, tag, (uint32_t)rel, 0u);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc_emit += __shfl_xor_sync(kFull, acc_emit, o);
    if (lane == 0 && acc_emit != 0.0) atomicAdd(&P.result->emitted, acc_emit);
    slab_epilogue(P.slab, false);
}

// internal accumulator -> caller's array: out[gid] += weight * acc[internal(gid)], acc reset to zero
struct UnpadParams {
    double *out, *acc;
    float *acc32;
    double weight;                      // ACC32: weight * e_ref
    int nx, ny, nbx, nby, nrp;
    long long n_root, n_total;
};

template <bool ACC32>
__global__ void __launch_bounds__(256) unpad_add_kernel(const __grid_constant__ UnpadParams U)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x; gid < U.n_total; gid += stride) {
        long long j;
        if (gid < U.n_root) {
            const int g = (int)gid;
            const int ix = g % U.nx, r = g / U.nx, iy = r % U.ny, iz = r / U.ny;
            const int X = ix + 2, Y = iy + 2, Z = iz + 2;
            j = 8ll * ((X >> 1) + U.nbx * ((Y >> 1) + (long long)U.nby * (Z >> 1))) + (X & 1) + 2 * (Y & 1) + 4 * (Z & 1);
        } else {
            j = U.nrp + (gid - U.n_root);
        }
        if (ACC32) {
            const float v = U.acc32[j];
            if (v != 0.0f) {
                U.out[gid] += U.weight * (double)v;
                U.acc32[j] = 0.0f;
            }
        } else {
            const double v = U.acc[j];
            if (v != 0.0) {
                U.out[gid] += U.weight * v;
                U.acc[j] = 0.0;
            }
        }
    }
}

// the hot-cell sums of a launch (FastParams::hot64) -> caller's array, sums reset to zero
struct HotFoldParams {
    double *out, *hot64;
    double weight;
    int nx, ny, nz, n_point, hot_r;
    int cell[SOC_MAX_POINT_SOURCES][3];          // root cell of every point source
};
__global__ void __launch_bounds__(256) hot_fold_kernel(const __grid_constant__ HotFoldParams H)
{
    const int side = 2 * H.hot_r + 1, cells = side * side * side;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < cells * H.n_point; i += gridDim.x * blockDim.x) {
        const double v = H.hot64[i];
        if (v == 0.0) continue;
        H.hot64[i] = 0.0;
        const int k = i / cells, j = i - k * cells;
        const int jz = j / (side * side), jr = j - jz * side * side, jy = jr / side, jx = jr - jy * side;
        const int ix = H.cell[k][0] + jx - H.hot_r, iy = H.cell[k][1] + jy - H.hot_r, iz = H.cell[k][2] + jz - H.hot_r;
        if ((unsigned)ix < (unsigned)H.nx && (unsigned)iy < (unsigned)H.ny && (unsigned)iz < (unsigned)H.nz)
            atomicAdd(H.out + (ix + (long long)H.nx * (iy + (long long)H.ny * iz)), H.weight * v);   // cubes of two sources may overlap
    }
}

// a11: energy balance by table lookup, 4 cells per thread, table in shared memory
struct TempParams {
    const uint32_t *cellw;
    const double *absorbed;
    const float *table;
    float *T_out;
    long long n_total;
    long long level_off[SOC_MAX_LEVELS + 1];
    int n_levels, n_table;
    double scale, e_min, e_max, inv_e_min;
    float x_scale;          // (n_table - 1) / ln(E_max / E_min)
};

__device__ __forceinline__ float temperature_of(const TempParams &P, const float *tab, uint32_t cw, double a, double inv_vol)
{
    if ((int32_t)cw < 0) return 0.0f;                       // parent cell
    const float rho = __uint_as_float(cw);
    if (!(rho > 0.0f)) return 0.0f;
    const double e = P.scale * a / (double)rho * inv_vol;
    if (!(e > P.e_min)) return tab[0];                      // also cells never hit
    if (e >= P.e_max) return tab[P.n_table - 1];
    const float x = logf((float)(e * P.inv_e_min)) * P.x_scale;
    int i = (int)x;
    i = i > P.n_table - 2 ? P.n_table - 2 : i;
    const float t0 = tab[i], t1 = tab[i + 1];
    return fmaf(x - (float)i, t1 - t0, t0);
}

__global__ void __launch_bounds__(256) temperature_kernel(const __grid_constant__ TempParams P)
{
    extern __shared__ float tab[];
    for (int i = threadIdx.x; i < P.n_table; i += blockDim.x) tab[i] = P.table[i];
    __syncthreads();
    const long long n4 = P.n_total >> 2;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n4 + 1; q += stride) {
        const long long c0 = q << 2;
        if (q < n4) {
            const uint4 cw = __ldg(reinterpret_cast<const uint4 *>(P.cellw) + q);
            const double2 a01 = __ldg(reinterpret_cast<const double2 *>(P.absorbed) + 2 * q);
            const double2 a23 = __ldg(reinterpret_cast<const double2 *>(P.absorbed) + 2 * q + 1);
            // the four cells may straddle a level boundary: find the inverse volume per cell
            double iv[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                int l = 0;
                while (l + 1 < P.n_levels && c0 + j >= P.level_off[l + 1]) ++l;
                iv[j] = (double)(1ull << (3 * l));
            }
            float4 t;
            t.x = temperature_of(P, tab, cw.x, a01.x, iv[0]);
            t.y = temperature_of(P, tab, cw.y, a01.y, iv[1]);
            t.z = temperature_of(P, tab, cw.z, a23.x, iv[2]);
            t.w = temperature_of(P, tab, cw.w, a23.y, iv[3]);
            reinterpret_cast<float4 *>(P.T_out)[q] = t;
        } else {
            for (long long c = c0; c < P.n_total; ++c) {     // ragged tail
                int l = 0;
                while (l + 1 < P.n_levels && c >= P.level_off[l + 1]) ++l;
                P.T_out[c] = temperature_of(P, tab, P.cellw[c], P.absorbed[c], (double)(1ull << (3 * l)));
            }
        }
    }
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}

// regular grid, every cell a leaf: density -> cell word in place (-0 -> +0, sign bit clear), validity flag and sum of
// the densities (soc_grid_create of large regular grids; small and hierarchical grids are converted on the host)
__global__ void __launch_bounds__(256) leafwords_kernel(uint32_t *cellw, long long n, double *sum_out, int *bad_out)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    double sum = 0.0;
    int bad = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const float r = __uint_as_float(cellw[i]);
        if (!(r >= 0.0f) || isinf(r)) bad = 1;
        cellw[i] = __float_as_uint(r + 0.0f) & 0x7fffffffu;
        sum += (double)r;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sum += __shfl_xor_sync(kFull, sum, o);
        bad |= __shfl_xor_sync(kFull, bad, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(sum_out, sum);
        if (bad) atomicOr(bad_out, 1);
    }
}

__global__ void __launch_bounds__(256) fill_i32_kernel(int32_t *a, long long n, int32_t v)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) a[i] = v;
}

// hierarchical grids of >= 2^20 cells: cell words, reverse links and validation on the GPU (soc_grid_create).  cellw holds
// the uploaded fp32 densities on entry.  flags: 1 bad density, 2 bad child index, 4 octet with two parents
struct HierParams {
    uint32_t *cellw;
    const int32_t *child;
    int32_t *parent;                    // [n_octets], preset to INT32_MIN
    long long n_total, n_root;
    int n_levels;
    long long level_off[SOC_MAX_LEVELS + 1];
    double *sum_out;                    // [0] sum of the root-leaf densities, [1] their number
    int *flags;
};

__global__ void __launch_bounds__(256) hierwords_kernel(const __grid_constant__ HierParams H)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    double sum = 0.0, cnt = 0.0;
    int bad = 0;
    for (long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x; gid < H.n_total; gid += stride) {
        int l = 0;
        while (l + 1 < H.n_levels && gid >= H.level_off[l + 1]) ++l;
        const int32_t ch = H.child[gid];
        if (ch < 0) {
            const float r = __uint_as_float(H.cellw[gid]);
            if (!(r >= 0.0f) || isinf(r)) bad |= 1;
            H.cellw[gid] = __float_as_uint(r + 0.0f) & 0x7fffffffu;
            if (gid < H.n_root) { sum += (double)r; cnt += 1.0; }
            continue;
        }
        if (l + 1 >= H.n_levels || (ch & 7) != 0 || (long long)ch + 8 > H.level_off[l + 2] - H.level_off[l + 1]) { bad |= 2; continue; }
        const long long child_rel = H.level_off[l + 1] + ch - H.n_root;
        if (atomicCAS(H.parent + (child_rel >> 3), INT32_MIN, (int32_t)(gid - H.n_root)) != INT32_MIN) bad |= 4;
        H.cellw[gid] = 0x80000000u | (uint32_t)child_rel;
    }
    sum = warp_sum(sum); cnt = warp_sum(cnt);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bad |= __shfl_xor_sync(kFull, bad, o);
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(H.sum_out, sum); atomicAdd(H.sum_out + 1, cnt);
        if (bad) atomicOr(H.flags, bad);
    }
}

// reverse links in the internal layout; flags |= 8 for an octet without a parent
__global__ void __launch_bounds__(256) parent_internal_kernel(const int32_t *parent, int32_t *pi, long long n_octets, int nx, int ny,
                                                              long long nbx, long long nby, long long nrp, long long n_root, int *flags)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < n_octets; o += stride) {
        const int32_t p = parent[o];
        if (p == INT32_MIN) { atomicOr(flags, 8); pi[o] = 0; continue; }
        const long long gid = (long long)p + n_root;
        long long j;
        if (gid >= n_root) j = nrp + (gid - n_root);
        else {
            const long long ix = gid % nx, r = gid / nx, iy = r % ny, iz = r / ny;
            const long long X = ix + 2, Y = iy + 2, Z = iz + 2;
            j = 8 * ((X >> 1) + nbx * ((Y >> 1) + nby * (Z >> 1))) + (X & 1) + 2 * (Y & 1) + 4 * (Z & 1);
        }
        pi[o] = (int32_t)j;
    }
}

// ABI-order cell words -> internal layout (ghost-padded 2x2x2 bricks of the root grid, then the octet levels with
// their links shifted behind the padded root grid); runs once per soc_grid_create
__global__ void __launch_bounds__(256) repad_kernel(const uint32_t *cellw, uint32_t *ci, int nx, int ny, int nz, int nbx,
                                                    int nby, long long nrp, long long n_root, long long n_int)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < n_int; j += stride) {
        uint32_t cw = kSentinel;
        bool real = true;
        if (j < nrp) {
            const long long B = j >> 3;
            const int slot = (int)(j & 7);
            const int bx = (int)(B % nbx), by = (int)((B / nbx) % nby), bz = (int)(B / ((long long)nbx * nby));
            const int ix = 2 * bx + (slot & 1) - 2, iy = 2 * by + ((slot >> 1) & 1) - 2, iz = 2 * bz + (slot >> 2) - 2;
            real = (unsigned)ix < (unsigned)nx && (unsigned)iy < (unsigned)ny && (unsigned)iz < (unsigned)nz;
            if (real) cw = cellw[ix + (long long)nx * (iy + (long long)ny * iz)];
        } else {
            cw = cellw[n_root + (j - nrp)];
        }
        if (real && (int32_t)cw < 0) cw = 0x80000000u | (uint32_t)(nrp + (cw & 0x7fffffffu));
        ci[j] = cw;
    }
}

__global__ void scale_kernel(double *a, long long n, double s)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) a[i] *= s;
}

// ------------------------------------------------------------------------------------------------
// f1: dust re-emission -- luminosities, package counts, prefix sums
// ------------------------------------------------------------------------------------------------
struct LumParams {
    const uint32_t *cellw;              // ABI order
    const float *T;
    double kabs, freq_hz;
    long long n_total;
    int n_levels;
    long long level_off[SOC_MAX_LEVELS + 1];
};

__device__ __forceinline__ double lum_of(const LumParams &L, long long c)
{
    int l = 0;
    while (l + 1 < L.n_levels && c >= L.level_off[l + 1]) ++l;
    return cell_luminosity(L.kabs, L.freq_hz, L.cellw[c], l, L.T[c]);
}

// out[0] += sum of L_c over all cells (count == NULL) or over the cells that send packages; out[1] += number of cells
// with L_c > 0
__global__ void __launch_bounds__(256) lum_sum_kernel(const __grid_constant__ LumParams L, const int32_t *count, double *out)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    double sum = 0.0, n_emit = 0.0;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < L.n_total; c += stride) {
        const double l = lum_of(L, c);
        if (l > 0.0 && (!count || count[c] > 0)) { sum += l; n_emit += 1.0; }
    }
    sum = warp_sum(sum); n_emit = warp_sum(n_emit);
    if ((threadIdx.x & 31) == 0) { atomicAdd(out, sum); atomicAdd(out + 1, n_emit); }
}

// package counts per cell: mode 0 the same number m from every emitting cell, mode 1 in proportion to the
// luminosity with a cap; out[2] += sum of the counts.  in[0] = sum L, in[1] = number of emitting cells
__global__ void __launch_bounds__(256) dust_counts_kernel(const __grid_constant__ LumParams L, int mode, long long n_request,
                                                          int cap, int32_t *count, double *scal)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    const double tot = scal[0];
    const long long n_emit = (long long)scal[1];
    const long long m = n_emit > 0 ? (n_request + n_emit - 1) / n_emit : 0;
    double n_sum = 0.0;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < L.n_total; c += stride) {
        const double l = lum_of(L, c);
        long long n = 0;
        if (l > 0.0 && n_request > 0) {
            if (mode == 0) n = m;
            else {
                n = (long long)ceil((double)n_request * l / tot);
                n = n < 1 ? 1 : (n > cap ? cap : n);
            }
        }
        count[c] = (int32_t)n;
        n_sum += (double)n;
    }
    n_sum = warp_sum(n_sum);
    if ((threadIdx.x & 31) == 0) atomicAdd(scal + 2, n_sum);
}

// exclusive prefix sums of count[n] -> first[n + 1], three passes over blocks of 2048 elements
constexpr int kScanBlock = 2048;

__global__ void __launch_bounds__(256) scan_block_sums_kernel(const int32_t *count, long long n, uint32_t *block_sums)
{
    __shared__ uint32_t s_w[8];
    const long long base = (long long)blockIdx.x * kScanBlock;
    uint32_t v = 0;
    for (int i = threadIdx.x; i < kScanBlock; i += 256) {
        const long long c = base + i;
        if (c < n) v += (uint32_t)count[c];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < 8; ++w) t += s_w[w];
        block_sums[blockIdx.x] = t;
    }
}

__global__ void __launch_bounds__(1024) scan_offsets_kernel(uint32_t *block_sums, int n_blocks)      // one block, in place
{
    __shared__ uint32_t s_part[1024];
    const int per = (n_blocks + 1023) / 1024;
    const int b0 = threadIdx.x * per, b1 = b0 + per < n_blocks ? b0 + per : n_blocks;
    uint32_t t = 0;
    for (int b = b0; b < b1; ++b) t += block_sums[b];
    s_part[threadIdx.x] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t run = 0;
        for (int i = 0; i < 1024; ++i) { const uint32_t v = s_part[i]; s_part[i] = run; run += v; }
    }
    __syncthreads();
    uint32_t run = s_part[threadIdx.x];
    for (int b = b0; b < b1; ++b) { const uint32_t v = block_sums[b]; block_sums[b] = run; run += v; }
}

__global__ void __launch_bounds__(256) scan_write_kernel(const int32_t *count, long long n, const uint32_t *block_offsets,
                                                         uint32_t *first)
{
    // thread t owns the 8 consecutive elements base + 8 t ..; warp and block scans of the per-thread sums
    __shared__ uint32_t s_w[8];
    const long long base = (long long)blockIdx.x * kScanBlock + 8ll * threadIdx.x;
    uint32_t v[8], sum = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { v[j] = base + j < n ? (uint32_t)count[base + j] : 0u; sum += v[j]; }
    uint32_t incl = sum;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(kFull, incl, o); if (lane >= o) incl += y; }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    uint32_t off = block_offsets[blockIdx.x];
    for (int w = 0; w < warp; ++w) off += s_w[w];
    uint32_t run = off + incl - sum;
#pragma unroll
    for (int j = 0; j < 8; ++j) { if (base + j < n) first[base + j] = run; run += v[j]; }
    if (base <= n - 1 && n - 1 < base + 8) first[n] = run;          // the thread that owns the last element closes the array
}

// f3: emitted[c] = sum_f w_f L_c,f(T_c)
__global__ void __launch_bounds__(256) cell_emission_kernel(const __grid_constant__ LumParams L, const double *freqtab,
                                                            int n_freq, double *emitted)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < L.n_total; c += stride) {
        int l = 0;
        while (l + 1 < L.n_levels && c >= L.level_off[l + 1]) ++l;
        const uint32_t cw = L.cellw[c];
        const float T = L.T[c];
        double sum = 0.0;
        if ((int32_t)cw >= 0 && __uint_as_float(cw) > 0.0f && T > 0.0f)
            for (int f = 0; f < n_freq; ++f)
                sum += freqtab[2 * n_freq + f] * cell_luminosity(freqtab[n_freq + f], freqtab[f], cw, l, T);
        emitted[c] = sum;
    }
}

// f3: effective absorbed energy of the diagonal ALI update: (A - S) / (1 - beta), beta = S / emitted in [0, 0.999]
__global__ void __launch_bounds__(256) ali_effective_kernel(const double *absorbed, const double *self_abs, const double *emitted,
                                                            long long n, double *eff)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += stride) {
        double beta = emitted[c] > 0.0 ? self_abs[c] / emitted[c] : 0.0;
        beta = beta > 0.999 ? 0.999 : (beta < 0.0 ? 0.0 : beta);
        const double e = (absorbed[c] - self_abs[c]) / (1.0 - beta);
        eff[c] = e < 0.0 ? 0.0 : e;
    }
}

// running mean of the reference field: r = (W r + n d) / (W + n) for up to three arrays at once
__global__ void __launch_bounds__(256) running_mean_kernel(double *r0, const double *d0, double *r1, const double *d1, double *r2,
                                                           const double *d2, long long n, double w_old, double w_new)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    const double inv = 1.0 / (w_old + w_new);
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += stride) {
        r0[c] = (w_old * r0[c] + w_new * d0[c]) * inv;
        if (r1) r1[c] = (w_old * r1[c] + w_new * d1[c]) * inv;
        if (r2) r2[c] = (w_old * r2[c] + w_new * d2[c]) * inv;
    }
}

__global__ void __launch_bounds__(256) add_kernel(double *out, const double *a, const double *b, long long n)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += stride) out[c] = a[c] + b[c];
}

// ------------------------------------------------------------------------------------------------
// f2: surface-brightness maps: one line of sight per thread, the cells walked as the packages walk
// them (a5 / a6) in fp64 on the ABI-order arrays; emission with extinction, front to back
// ------------------------------------------------------------------------------------------------
struct MapParams {
    int nx, ny, nz, n_root, hier;
    const uint32_t *cellw;
    const int32_t *parent;
    const float *T;
    double kabs, ksca, freq_hz;
    double ex[3], ey[3], dir[3], centre[3];
    int npx, npy;
    double pixel;
    float *map;
};

__global__ void __launch_bounds__(128) map_kernel(const __grid_constant__ MapParams M)
{
    const long long n_pix = (long long)M.npx * M.npy;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const double N[3] = {(double)M.nx, (double)M.ny, (double)M.nz};
    const int n_i[3] = {M.nx, M.ny, M.nz};
    const double kext = M.kabs + M.ksca;
    const double inf = __longlong_as_double(0x7ff0000000000000ll);
    for (long long pix = (long long)blockIdx.x * blockDim.x + threadIdx.x; pix < n_pix; pix += stride) {
        const int i = (int)(pix % M.npx), j = (int)(pix / M.npx);
        const double a = ((double)i + 0.5 - 0.5 * (double)M.npx) * M.pixel, b = ((double)j + 0.5 - 0.5 * (double)M.npy) * M.pixel;
        double o[3], t_in = -inf, t_out = inf;
#pragma unroll
        for (int k = 0; k < 3; ++k) o[k] = M.centre[k] + a * M.ex[k] + b * M.ey[k];
#pragma unroll
        for (int k = 0; k < 3; ++k) {                        // slab test against [0, N_k]
            if (M.dir[k] != 0.0) {
                double t0 = (0.0 - o[k]) / M.dir[k], t1 = (N[k] - o[k]) / M.dir[k];
                if (t0 > t1) { const double t = t0; t0 = t1; t1 = t; }
                t_in = t0 > t_in ? t0 : t_in;
                t_out = t1 < t_out ? t1 : t_out;
            } else if (o[k] < 0.0 || o[k] > N[k]) t_in = inf;
        }
        double I = 0.0, tau = 0.0;
        if (t_in < t_out) {
            int c3[3];
            double f[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double x = o[k] + t_in * M.dir[k];
                int c = (int)floor(x);
                c = c < 0 ? 0 : (c > n_i[k] - 1 ? n_i[k] - 1 : c);
                double fk = x - (double)c;
                f[k] = fk < 0.0 ? 0.0 : (fk > 1.0 ? 1.0 : fk);
                c3[k] = c;
            }
            int rel = c3[0] + M.nx * (c3[1] + M.ny * c3[2]);            // root cell id; octet cells: id of the ABI vector
            int lev = 0;                                              // level - 1
            bool inside = true;
            while (inside) {
                // a6: down to the leaf that holds the position
                uint32_t cw = __ldg(M.cellw + rel);
                while ((int32_t)cw < 0) {
                    int slot = 0;
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        if (f[k] >= 0.5) { slot |= 1 << k; f[k] = 2.0 * f[k] - 1.0; } else f[k] = 2.0 * f[k];
                    }
                    rel = M.n_root + (int)(cw & 0x7fffffffu) + slot;
                    lev += 1;
                    cw = __ldg(M.cellw + rel);
                }
                double t[3];
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const double d = M.dir[k];
                    double tk = d > 0.0 ? (1.0 - f[k]) / d : (d < 0.0 ? (-f[k]) / d : inf);
                    t[k] = tk < 0.0 ? 0.0 : tk;
                }
                int ax = 0;                                  // lowest axis wins a tie (S4)
                if (t[1] < t[ax]) ax = 1;
                if (t[2] < t[ax]) ax = 2;
                const double ts = t[ax];
                const double ds = ts / (double)(1 << lev);
                const double dtau = kext * (double)__uint_as_float(cw) * ds;
                const double Tc = (double)__ldg(M.T + rel);
                if (dtau > 0.0 && Tc > 0.0) I += exp(-tau) * (M.kabs / kext) * planck_nu(M.freq_hz, Tc) * (-expm1(-dtau));
                tau += dtau;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const double fn = f[k] + ts * M.dir[k];
                    f[k] = fn < 0.0 ? 0.0 : (fn > 1.0 ? 1.0 : fn);
                }
                // a5 / a6: across the face of axis ax -- sibling flip, else up to the common parent
                const int sg = M.dir[ax] > 0.0 ? 1 : -1;
                bool found = false;
                while (lev > 0) {
                    const int oct = rel - M.n_root;
                    const int bit = (oct >> ax) & 1;
                    if ((sg > 0) != (bit != 0)) { rel ^= (1 << ax); found = true; break; }
#pragma unroll
                    for (int k = 0; k < 3; ++k) f[k] = (f[k] + (double)((oct >> k) & 1)) * 0.5;
                    const int par = __ldg(M.parent + (oct >> 3));             // parent id - n_root (negative: a root cell)
                    rel = par + M.n_root;
                    lev -= 1;
                }
                if (!found) {
                    int ix = rel % M.nx, iy = (rel / M.nx) % M.ny, iz = rel / (M.nx * M.ny);
                    if (ax == 0) ix += sg; else if (ax == 1) iy += sg; else iz += sg;
                    if ((unsigned)ix >= (unsigned)M.nx || (unsigned)iy >= (unsigned)M.ny || (unsigned)iz >= (unsigned)M.nz) inside = false;
                    rel = ix + M.nx * (iy + M.ny * iz);
                }
                f[ax] = sg > 0 ? 0.0 : 1.0;
            }
        }
        M.map[pix] = (float)I;
    }
}

// ------------------------------------------------------------------------------------------------
// f4: stochastically heated grains.  One CTA per cell, its warps take the grain sizes in turn; per
// (cell, size) a warp builds the upward rates in a shared tile (a lane owns the columns lane, lane + 32, ...: no atomics),
// turns every column into its suffix sums B_ji = sum_{k >= j} R_ki, and runs the forward substitution on the probability
// flux across the bin boundaries,  p_j = (sum_{i < j} p_i B_ji) / R_(j-1,j)  -- all terms positive, the sums in fp64 (the
// paper: "worked reliably but only when part of the operations were performed in double precision").
// ------------------------------------------------------------------------------------------------
struct StochParams {
    int n_size, n_e, n_freq, warps;
    const int32_t *jupT;                // [n_size][n_freq][n_e]
    const float *wupT;                  // [n_size][n_freq][n_e]
    const double *cool;                 // [n_size][n_e]
    const float *emis;                  // [n_size][n_e][n_freq], scaled by emis_scale[s] to stay inside fp32
    const double *emis_scale;           // [n_size] abundance[s] / scale of emis
    const double *intensity;
    long long n_cells;
    double *emission, *p_out;
};

__global__ void __launch_bounds__(128) stochastic_kernel(const __grid_constant__ StochParams S)
{
    extern __shared__ double s_mem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ne = S.n_e, nf = S.n_freq;
    double *s_int = s_mem;                                         // [nf] intensities of this cell
    double *s_em = s_int + nf + (size_t)warp * (nf + ne);          // [nf] this warp's emission sums
    double *s_p = s_em + nf;                                       // [ne]
    float *s_tile = reinterpret_cast<float *>(s_mem + nf + (size_t)S.warps * (nf + ne)) + (size_t)warp * ne * ne;   // [ne][ne]
    for (long long cell = blockIdx.x; cell < S.n_cells; cell += gridDim.x) {
        __syncthreads();
        for (int f = threadIdx.x; f < nf; f += blockDim.x) s_int[f] = S.intensity[cell * nf + f];
        for (int f = lane; f < nf; f += 32) s_em[f] = 0.0;
        __syncthreads();
        for (int sz = warp; sz < S.n_size; sz += S.warps) {
            for (int k = lane; k < ne * ne; k += 32) s_tile[k] = 0.0f;
            __syncwarp();
            // upward rates: R_ji += w_jif I_f, column i owned by one lane
            const int32_t *jt = S.jupT + (size_t)sz * nf * ne;
            const float *wt = S.wupT + (size_t)sz * nf * ne;
            for (int i = lane; i < ne; i += 32)
                for (int f = 0; f < nf; ++f) {
                    const int j = __ldg(jt + (size_t)f * ne + i);
                    if (j >= 0) s_tile[j * ne + i] += (float)((double)__ldg(wt + (size_t)f * ne + i) * s_int[f]);
                }
            // suffix sums down every column: B_ji = sum_{k >= j} R_ki
            for (int i = lane; i < ne; i += 32) {
                float run = 0.0f;
                for (int j = ne - 1; j > i; --j) { run += s_tile[j * ne + i]; s_tile[j * ne + i] = run; }
            }
            __syncwarp();
            // forward substitution, p_0 = 1, rescaled when it grows out of range
            const double *cool = S.cool + (size_t)sz * ne;
            if (lane == 0) s_p[0] = 1.0;
            __syncwarp();
            for (int j = 1; j < ne; ++j) {
                double acc = 0.0;
                for (int i = lane; i < j; i += 32) acc += s_p[i] * (double)s_tile[j * ne + i];
                acc = warp_sum(acc);
                double pj = acc / cool[j];
                if (pj > 1e200) {                                  // warp-uniform
                    for (int i = lane; i < j; i += 32) s_p[i] *= 1e-200;
                    pj *= 1e-200;
                }
                __syncwarp();
                if (lane == 0) s_p[j] = pj;
                __syncwarp();
            }
            double tot = 0.0;
            for (int i = lane; i < ne; i += 32) tot += s_p[i];
            tot = warp_sum(tot);
            const double inv = 1.0 / tot;
            for (int i = lane; i < ne; i += 32) {
                const double p = s_p[i] * inv;
                s_p[i] = p;
                if (S.p_out) S.p_out[((size_t)cell * S.n_size + sz) * ne + i] = p;
            }
            __syncwarp();
            // emission of this size: sum_i p_i emis_if
            const float *em = S.emis + (size_t)sz * ne * nf;
            const double sc = S.emis_scale[sz];
            for (int f = lane; f < nf; f += 32) {
                double e = 0.0;
                for (int i = 0; i < ne; ++i) e += s_p[i] * (double)__ldg(em + (size_t)i * nf + f);
                s_em[f] += sc * e;
            }
            __syncwarp();
        }
        __syncthreads();
        for (int f = threadIdx.x; f < nf; f += blockDim.x) {
            double e = 0.0;
            for (int w = 0; w < S.warps; ++w) e += s_mem[nf + (size_t)w * (nf + ne) + f];
            S.emission[cell * nf + f] = e;
        }
    }
}

// roofline probes: random gathers / random reductions over a footprint
__device__ __forceinline__ uint32_t mix32(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

constexpr int kProbeHotMax = 8192;      // cells of the shared-memory hot-spot probe (kind 7)

template <int KIND>
__global__ void __launch_bounds__(256) probe_kernel(void *buf, unsigned long long n_elem, long long ops_per_thread, float *sink)
{
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t s = mix32(tid * 2654435761u + 12345u);
    float acc[4] = {0.f, 0.f, 0.f, 0.f};          // four independent chains: four gathers in flight per thread
    // KIND 7: the remedy the photon kernels use for the cells around a point source -- the block's partial sums in shared
    // memory, one fp64 reduction per cell and block at the end (n_elem <= kProbeHotMax)
    __shared__ float s_hot[KIND == 7 ? kProbeHotMax : 1];
    if (KIND == 7) {
        for (unsigned i = threadIdx.x; i < n_elem; i += blockDim.x) s_hot[i] = 0.0f;
        __syncthreads();
    }
    for (long long i = 0; i < ops_per_thread; i += 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            s = mix32(s + 0x9e3779b9u);
            const unsigned long long j = ((unsigned long long)s * n_elem) >> 32;
            if (KIND == 0) acc[u] += __ldg(reinterpret_cast<const float *>(buf) + j);
            else if (KIND == 1) atomicAdd(reinterpret_cast<double *>(buf) + j, 1.0);
            else if (KIND == 2) atomicAdd(reinterpret_cast<float *>(buf) + j, 1.0f);
            else if (KIND == 3) {                // 32-byte gather (one sector: a 2x2x2 brick of fp32 cells)
                float a0, a1, a2, a3, a4, a5, a6, a7;
                asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                             : "=f"(a0), "=f"(a1), "=f"(a2), "=f"(a3), "=f"(a4), "=f"(a5), "=f"(a6), "=f"(a7)
                             : "l"(reinterpret_cast<const float *>(buf) + 8 * j));
                acc[u] += a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
            } else if (KIND == 4) {              // 16-byte vector reduction (4 fp32 cells)
                asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(reinterpret_cast<float *>(buf) + 4 * j),
                             "f"(1.0f), "f"(1.0f), "f"(1.0f), "f"(1.0f) : "memory");
            } else if (KIND == 7) {
                atomicAdd(s_hot + j, 1.0f);
            } else if (KIND == 6) {              // 16-byte gather (half a brick: what photon_q_kernel loads)
                const uint4 v = __ldg(reinterpret_cast<const uint4 *>(buf) + j);
                acc[u] += __uint_as_float(v.x ^ v.y ^ v.z ^ v.w);
            } else {                             // the memory side of one cell-step: gather rho[cell], add to acc[cell]
                acc[u] += __ldg(reinterpret_cast<const float *>(buf) + j);
                atomicAdd(reinterpret_cast<float *>(buf) + n_elem + j, 1.0f);
            }
        }
    }
    if ((KIND == 0 || KIND == 3 || KIND == 5 || KIND == 6) && acc[0] + acc[1] + acc[2] + acc[3] == 123.456f) *sink = acc[0];
    if (KIND == 7) {
        __syncthreads();
        for (unsigned i = threadIdx.x; i < n_elem; i += blockDim.x)
            if (s_hot[i] != 0.0f) atomicAdd(reinterpret_cast<double *>(buf) + i, (double)s_hot[i]);
    }
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------------
namespace {

int ensure_slots(soc_grid *G, int n)
{
    if (n <= G->n_slots) return SOC_OK;
    if (G->d_results) cudaFree(G->d_results);
    if (G->d_counters) cudaFree(G->d_counters);
    if (G->h_results) cudaFreeHost(G->h_results);
    G->d_results = nullptr; G->d_counters = nullptr; G->h_results = nullptr; G->n_slots = 0;
    SOC_CUDA(cudaMalloc(&G->d_results, sizeof(DevResult) * n));
    SOC_CUDA(cudaMalloc(&G->d_counters, sizeof(unsigned long long) * n));
    SOC_CUDA(cudaMallocHost(&G->h_results, sizeof(DevResult) * n));
    G->n_slots = n;
    return SOC_OK;
}

int ensure_events(soc_grid *G, int n)
{
    while ((int)G->ev0.size() < n) {
        cudaEvent_t a, b;
        SOC_CUDA(cudaEventCreate(&a));
        SOC_CUDA(cudaEventCreate(&b));
        G->ev0.push_back(a); G->ev1.push_back(b); G->ev_set.push_back(0);
    }
    return SOC_OK;
}

template <typename K> int blocks_for(soc_grid *G, K kernel, int threads, int *blocks)
{
    int per_sm = 0;
    SOC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, 0));
    if (per_sm < 1) return fail(SOC_ECUDA, "photon kernel does not fit on an SM");
    if (G->opt_blocks_per_sm > 0 && G->opt_blocks_per_sm < per_sm) per_sm = G->opt_blocks_per_sm;
    *blocks = per_sm * G->n_sm;                 // persistent: a whole number of CTAs per SM
    return SOC_OK;
}

template <typename R, bool HIER, bool REPLAY> int launch_photon(soc_grid *G, const SimParams &P, cudaStream_t st)
{
    int blocks = 0;
    const int threads = G->opt_threads;
    int rc = blocks_for(G, photon_kernel<R, HIER, REPLAY>, threads, &blocks);
    if (rc != SOC_OK) return rc;
    // do not launch more lanes than there are packages (rounded up to whole blocks)
    const long long n_pkg = P.pkg_end - P.pkg_begin;
    const long long need = (n_pkg + threads - 1) / threads;
    if (need < blocks) blocks = (int)(need > 0 ? need : 1);
    photon_kernel<R, HIER, REPLAY><<<blocks, threads, 0, st>>>(P);
    g_launches += 1;
    SOC_CUDA(cudaGetLastError());
    return SOC_OK;
}

// the hot-cell sums of the launch described by P follow the internal accumulator into the caller's array
int launch_hot_fold(soc_grid *G, const FastParams &P, double weight, double *absorbed, cudaStream_t st)
{
    if (P.hot_r < 0 || P.n_point <= 0 || !P.hot64) return SOC_OK;
    HotFoldParams H;
    std::memset(&H, 0, sizeof(H));
    H.out = absorbed; H.hot64 = P.hot64; H.weight = weight;
    H.nx = G->nx; H.ny = G->ny; H.nz = G->nz; H.n_point = P.n_point; H.hot_r = P.hot_r;
    for (int k = 0; k < P.n_point; ++k)
        for (int j = 0; j < 3; ++j) H.cell[k][j] = (int)std::floor(P.ps_pos[k][j]);
    const int side = 2 * P.hot_r + 1, n = side * side * side * P.n_point;
    hot_fold_kernel<<<(n + 255) / 256, 256, 0, st>>>(H);
    g_launches += 1;
    SOC_CUDA(cudaGetLastError());
    if (G->overlap_active) SOC_CUDA(cudaEventRecord(G->ev_unpad[G->acc_sel], st));    // the fold into the caller's array ends here
    return SOC_OK;
}

int launch_unpad(soc_grid *G, bool acc32, double weight, double *absorbed, cudaStream_t st)
{
    UnpadParams U;
    U.out = absorbed; U.acc = G->acc_sel ? G->d_acc_b : G->d_acc; U.acc32 = G->acc_sel ? G->d_acc32_b : G->d_acc32; U.weight = weight;
    if (G->unpad_wait) SOC_CUDA(cudaStreamWaitEvent(st, G->unpad_wait, 0));     // folds into the caller's array one at a time
    U.nx = G->nx; U.ny = G->ny; U.nbx = G->nbx; U.nby = G->nby; U.nrp = G->nrp;
    U.n_root = G->n_root; U.n_total = G->n_total;
    long long ub = (G->n_total + 255) / 256;
    const long long cap = (long long)G->n_sm * 8;
    if (ub > cap) ub = cap;
    if (acc32) unpad_add_kernel<true><<<(int)ub, 256, 0, st>>>(U);
    else unpad_add_kernel<false><<<(int)ub, 256, 0, st>>>(U);
    g_launches += 1;
    SOC_CUDA(cudaGetLastError());
    if (G->overlap_active) {
        SOC_CUDA(cudaEventRecord(G->ev_unpad[G->acc_sel], st));
        G->unpad_wait = G->ev_unpad[G->acc_sel];
    }
    return SOC_OK;
}

template <bool HIER, bool REPLAY, bool ACC32, bool QK, bool DUST, bool GROUP = false>
int launch_fast(soc_grid *G, const FastParams &P, double weight, double *absorbed, cudaStream_t st)
{
    static_assert(!(HIER && QK) && (ACC32 || !QK), "photon_q_kernel walks regular grids with the fp32 accumulator only");
    int blocks = 0;
    const int threads = G->opt_threads;
    const int side = 2 * P.hot_r + 1;
    const size_t smem = P.hot_r >= 0 ? sizeof(float) * (size_t)side * side * side * (size_t)P.n_point : 0;
    int per_sm = 0;
    if (QK) SOC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, photon_q_kernel<REPLAY, DUST, false>, threads, smem));
    else SOC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, photon_fast_kernel<HIER, REPLAY, ACC32, DUST, GROUP>, threads, smem));
    if (per_sm < 1) return fail(SOC_ECUDA, "photon kernel does not fit on an SM");
    if (G->opt_blocks_per_sm > 0 && G->opt_blocks_per_sm < per_sm) per_sm = G->opt_blocks_per_sm;
    blocks = per_sm * G->n_sm;                   // persistent: a whole number of CTAs per SM
    const long long n_pkg = P.pkg_end - P.pkg_begin;
    const long long need = (n_pkg + threads - 1) / threads;
    if (need < blocks) blocks = (int)(need > 0 ? need : 1);
    if (G->opt_carveout >= 0) {
        if (QK) SOC_CUDA(cudaFuncSetAttribute(photon_q_kernel<REPLAY, DUST, false>, cudaFuncAttributePreferredSharedMemoryCarveout, G->opt_carveout));
        else SOC_CUDA(cudaFuncSetAttribute(photon_fast_kernel<HIER, REPLAY, ACC32, DUST, GROUP>, cudaFuncAttributePreferredSharedMemoryCarveout, G->opt_carveout));
    }
    if (QK) photon_q_kernel<REPLAY, DUST, false><<<blocks, threads, smem, st>>>(P);
    else photon_fast_kernel<HIER, REPLAY, ACC32, DUST, GROUP><<<blocks, threads, smem, st>>>(P);
    g_launches += 1;
    SOC_CUDA(cudaGetLastError());
    if (G->ev_after_photon) {                    // "timing": the pair brackets the photon kernel alone
        SOC_CUDA(cudaEventRecord(G->ev_after_photon, st));
        G->ev_after_photon = nullptr;
    }
    const int rc = launch_unpad(G, ACC32, weight, absorbed, st);
    return rc == SOC_OK && ACC32 ? launch_hot_fold(G, P, weight, absorbed, st) : rc;
}

// Slab-blocked launch of one frequency on a regular grid (SlabParams): create the packages, sweep the z-slabs up and down
// `sweeps` times with photon_q_kernel<., ., SLAB> confined to one slab per launch, then one whole-grid launch that takes
// what is still queued (packages that scattered back across a slab boundary after the last sweep).
// `last`: the launch ends the frequency (a frequency of more than 2^24 packages is served in several such launches): the
// internal accumulator is folded into the caller's array.
template <bool STATS, bool DUST>
int launch_slab(soc_grid *G, FastParams P, int n_slabs, int sweeps, double weight, double *absorbed, bool last, cudaStream_t st)
{
    const int sel = G->acc_sel;
    const int threads = 256;
    const unsigned n_pkg = (unsigned)(P.pkg_end - P.pkg_begin);
    const int side = 2 * P.hot_r + 1;
    const size_t smem = P.hot_r >= 0 ? sizeof(float) * (size_t)side * side * side * (size_t)P.n_point : 0;
    int per_sm = 0;
    SOC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, photon_q_kernel<STATS, DUST, true>, threads, smem));
    if (per_sm < 1) return fail(SOC_ECUDA, "photon kernel does not fit on an SM");
    if (G->opt_blocks_per_sm > 0 && G->opt_blocks_per_sm < per_sm) per_sm = G->opt_blocks_per_sm;
    int blocks = per_sm * G->n_sm;
    const long long need = ((long long)n_pkg + threads - 1) / threads;
    if (need < blocks) blocks = (int)(need > 0 ? need : 1);
    // the phases: sweeps up and down over the slabs (an upward sweep ends at the top slab, the next starts just below it)
    std::vector<int> phase;
    for (int sweep = 0, s = 0, dir = 1; sweep < sweeps; ++sweep) {
        for (;; s += dir) {
            phase.push_back(s);
            if (s + dir < 0 || s + dir >= n_slabs) break;
        }
        dir = -dir;
        s += dir;
    }
    // queues: one per slab (every package of the launch may wait in one slab), two leftover queues (each receives, every
    // other phase, at most the packages the lanes hold)
    const size_t lanes = (size_t)blocks * threads;
    const size_t cap_left = (lanes < n_pkg ? lanes : n_pkg) * (phase.size() / 2 + 1);
    const size_t entries = (size_t)n_slabs * n_pkg + 2 * cap_left;
    if (cap_left >= (1ull << 32)) return fail(SOC_EINVAL, "too many phases");
    if (G->slab_q_entries[sel] < entries) {
        if (G->d_slab_q[sel]) { SOC_CUDA(cudaStreamSynchronize(st)); SOC_CUDA(cudaFree(G->d_slab_q[sel])); G->d_slab_q[sel] = nullptr; }
        G->slab_q_entries[sel] = 0;
        // a buffer left by an earlier grid of this process, if one is large enough (the smallest such)
        int best = -1;
        {
            std::lock_guard<std::mutex> lock(g_queue_cache_mutex);
            for (size_t i = 0; i < g_queue_cache.size(); ++i)
                if (g_queue_cache[i].device == G->device && g_queue_cache[i].entries >= entries &&
                    (best < 0 || g_queue_cache[i].entries < g_queue_cache[best].entries)) best = (int)i;
            if (best >= 0) {
                G->d_slab_q[sel] = (uint4 *)g_queue_cache[best].ptr;
                G->slab_q_entries[sel] = g_queue_cache[best].entries;
                g_queue_cache.erase(g_queue_cache.begin() + best);
            }
        }
        if (best < 0) {
            cudaError_t e = cudaMalloc(&G->d_slab_q[sel], entries * kQueueEntryBytes);
            if (e == cudaErrorMemoryAllocation) {           // idle buffers of the caches first, then once more
                cudaGetLastError();
                if (release_caches() > 0) e = cudaMalloc(&G->d_slab_q[sel], entries * kQueueEntryBytes);
            }
            if (e != cudaSuccess) {
                cudaGetLastError();
                G->d_slab_q[sel] = nullptr;
                return fail(SOC_ENOMEM, "package queues of the slab-blocked launch");
            }
            G->slab_q_entries[sel] = entries;
        }
    }
    const size_t stride = G->slab_q_entries[sel];    // the three arrays of the buffer are `stride` entries apart
    const size_t cnt_bytes = sizeof(unsigned) * kSlabCntLen;
    if (!G->d_slab_cnt[sel]) SOC_CUDA(cudaMalloc(&G->d_slab_cnt[sel], cnt_bytes));
    SlabParams &S = P.slab;
    S.qa = G->d_slab_q[sel]; S.qb = S.qa + stride; S.qc = S.qb + stride; S.qp = reinterpret_cast<float *>(S.qc + stride);
    S.cnt = G->d_slab_cnt[sel]; S.cap = n_pkg; S.cap_left = (unsigned)cap_left; S.n_slabs = n_slabs;
    S.limit = S.cap; S.limit_left = S.cap_left; S.q_entries = stride;
    if (G->opt_slab_queue_limit > 0) {
        if ((unsigned long long)G->opt_slab_queue_limit < S.limit) S.limit = (unsigned)G->opt_slab_queue_limit;
        if ((unsigned long long)G->opt_slab_queue_limit < S.limit_left) S.limit_left = (unsigned)G->opt_slab_queue_limit;
    }
    S.slab_ids = ((G->nbz + n_slabs - 1) / n_slabs) * 8 * G->nbx * G->nby;
    SOC_CUDA(cudaMemsetAsync(S.cnt, 0, cnt_bytes, st));
    {
        long long eb = ((long long)n_pkg + 255) / 256;
        const long long cap = (long long)G->n_sm * 16;
        S.q_left = n_slabs; S.s_first = 0; S.s_last = -1; S.final_phase = 0;
        slab_emit_kernel<<<(int)(eb < cap ? eb : cap), 256, 0, st>>>(P);
        g_launches += 1;
    }
    for (size_t k = 0; k < phase.size(); ++k) {
        S.s_first = S.s_last = phase[k];
        S.q_left = n_slabs + (int)(k & 1);
        photon_q_kernel<STATS, DUST, true><<<blocks, threads, smem, st>>>(P);
        g_launches += 1;
    }
    S.s_first = 0; S.s_last = n_slabs - 1; S.q_left = n_slabs + (int)(phase.size() & 1); S.final_phase = 1;
    photon_q_kernel<STATS, DUST, true><<<blocks, threads, smem, st>>>(P);
    g_launches += 1;
    SOC_CUDA(cudaGetLastError());
    if (!last) return SOC_OK;
    if (G->ev_after_photon) {
        SOC_CUDA(cudaEventRecord(G->ev_after_photon, st));
        G->ev_after_photon = nullptr;
    }
    const int rc = launch_unpad(G, true, weight, absorbed, st);
    return rc == SOC_OK ? launch_hot_fold(G, P, weight, absorbed, st) : rc;
}

// ---- f1 host helpers
void fill_lum_params(const soc_grid *G, int ifreq, const float *T, LumParams *L)
{
    std::memset(L, 0, sizeof(*L));
    L->cellw = G->d_cellw; L->T = T; L->kabs = G->kabs[ifreq]; L->freq_hz = G->freq[ifreq];
    L->n_total = G->n_total; L->n_levels = G->n_levels;
    for (int l = 0; l <= G->n_levels; ++l) L->level_off[l] = G->level_off[l];
}

int ensure_dust_buffers(soc_grid *G)
{
    if (G->d_dust_first) return SOC_OK;
    const long long n_blocks = (G->n_total + kScanBlock - 1) / kScanBlock;
    SOC_CUDA(cudaMalloc(&G->d_dust_first, sizeof(uint32_t) * (size_t)(G->n_total + 1)));
    SOC_CUDA(cudaMalloc(&G->d_scan_blocks, sizeof(uint32_t) * (size_t)n_blocks));
    SOC_CUDA(cudaMalloc(&G->d_scalars, sizeof(double) * 8));
    SOC_CUDA(cudaMallocHost(&G->h_scalars, sizeof(double) * 8));
    return SOC_OK;
}

// stride that spreads consecutive dust package ids over the cells: the odd number nearest below n / golden ratio that
// is coprime to n, so that q -> q * stride mod n is a permutation of [0, n)
unsigned long long dust_stride(long long n)
{
    if (n <= 2) return 1;
    long long s = (long long)std::floor((double)n * 0.6180339887498949) | 1;
    for (;;) {
        long long a = s, b = n;
        while (b) { const long long t = a % b; a = b; b = t; }
        if (a == 1) return (unsigned long long)s;
        s += 2;
    }
}

// prefix sums of the caller's package counts, sum of the luminosities of the sending cells; fills D.  Synchronises `st`.
int dust_prepare(soc_grid *G, int ifreq, const soc_sources *src, long long n_const, double weight, DustParams *D,
                 double *lum_total, cudaStream_t st)
{
    if (!src->dust_T || !src->dust_count) return fail(SOC_EINVAL, "dust packages requested but dust_T / dust_count is NULL");
    if (src->n_dust >= (1ll << 32)) return fail(SOC_EINVAL, "n_dust must be < 2^32");
    int rc = ensure_dust_buffers(G);
    if (rc != SOC_OK) return rc;
    LumParams L;
    fill_lum_params(G, ifreq, src->dust_T, &L);
    const int n_blocks = (int)((G->n_total + kScanBlock - 1) / kScanBlock);
    SOC_CUDA(cudaMemsetAsync(G->d_scalars, 0, sizeof(double) * 8, st));
    lum_sum_kernel<<<G->n_sm * 8, 256, 0, st>>>(L, src->dust_count, G->d_scalars);
    scan_block_sums_kernel<<<n_blocks, 256, 0, st>>>(src->dust_count, G->n_total, G->d_scan_blocks);
    scan_offsets_kernel<<<1, 1024, 0, st>>>(G->d_scan_blocks, n_blocks);
    scan_write_kernel<<<n_blocks, 256, 0, st>>>(src->dust_count, G->n_total, G->d_scan_blocks, G->d_dust_first);
    g_launches += 4;
    SOC_CUDA(cudaGetLastError());
    uint32_t total = 0;
    SOC_CUDA(cudaMemcpyAsync(G->h_scalars, G->d_scalars, sizeof(double) * 2, cudaMemcpyDeviceToHost, st));
    SOC_CUDA(cudaMemcpyAsync(&total, G->d_dust_first + G->n_total, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
    SOC_CUDA(cudaStreamSynchronize(st));
    if ((long long)total != src->n_dust) return fail(SOC_EINVAL, "n_dust is not the sum of dust_count");
    *lum_total = G->h_scalars[0];
    if (!(*lum_total > 0.0) || !std::isfinite(*lum_total)) return fail(SOC_EINVAL, "dust packages requested from cells that emit nothing");
    D->n_const = n_const; D->n_dust = src->n_dust; D->stride = dust_stride(src->n_dust);
    D->first = G->d_dust_first; D->count = src->dust_count; D->T = src->dust_T; D->self_abs = src->dust_self;
    D->kabs = G->kabs[ifreq]; D->freq_hz = G->freq[ifreq]; D->weight = weight;
    D->n_levels = G->n_levels;
    for (int l = 0; l <= G->n_levels; ++l) D->level_off[l] = (int)G->level_off[l];
    return SOC_OK;
}

int check_sources(const soc_grid *G, const soc_sources *src, long long n_packages, long long *n_bg_out)
{
    if (!src) return fail(SOC_EINVAL, "sources is NULL");
    if (src->beam) {
        for (int j = 0; j < 6; ++j)
            if (!std::isfinite(src->beam[j])) return fail(SOC_EINVAL, "beam is not finite");
        const int n[3] = {G->nx, G->ny, G->nz};
        for (int j = 0; j < 3; ++j)
            if (src->beam[j] < 0.0 || src->beam[j] > n[j]) return fail(SOC_EINVAL, "beam starts outside the grid");
        *n_bg_out = 0;
        return SOC_OK;
    }
    if (src->n_point < 0 || src->n_point > SOC_MAX_POINT_SOURCES) return fail(SOC_EINVAL, "n_point out of range");
    if (src->n_point > 0 && (!src->ps_pos || !src->ps_lum)) return fail(SOC_EINVAL, "point source arrays are NULL");
    const bool has_bg = src->bg_intensity > 0.0, has_ps = src->n_point > 0;
    if (src->n_dust < 0 || src->n_dust > n_packages) return fail(SOC_EINVAL, "n_dust out of range");
    const long long n_const = n_packages - src->n_dust;      // the dust packages are the last n_dust ids
    long long n_bg = src->n_bg;
    if (n_bg < 0) n_bg = (has_bg && has_ps) ? n_const / 2 : (has_bg ? n_const : 0);
    if (n_bg > n_const) return fail(SOC_EINVAL, "n_bg > n_packages - n_dust");
    if (n_bg > 0 && !(has_bg && std::isfinite(src->bg_intensity)))
        return fail(SOC_EINVAL, "background packages requested but bg_intensity <= 0");
    if (n_const - n_bg > 0 && !has_ps) return fail(SOC_EINVAL, "point-source packages requested but n_point == 0");
    for (int k = 0; k < src->n_point; ++k) {
        const double *q = src->ps_pos + 3 * k;
        if (!(q[0] > 0.0 && q[0] < G->nx && q[1] > 0.0 && q[1] < G->ny && q[2] > 0.0 && q[2] < G->nz))
            return fail(SOC_EINVAL, "point source outside the root grid");
        if (!(src->ps_lum[k] >= 0.0) || !std::isfinite(src->ps_lum[k])) return fail(SOC_EINVAL, "bad point source luminosity");
    }
    *n_bg_out = n_bg;
    return SOC_OK;
}

// enqueue one frequency into result slot `slot`
int enqueue_frequency(soc_grid *G, int ifreq, const soc_sources *src, long long n_packages, unsigned long long seed,
                      double weight, long long pkg_begin, long long pkg_count, double *absorbed,
                      soc_replay_record *replay, uint32_t flags, int slot, cudaStream_t st)
{
    if (!G) return fail(SOC_EINVAL, "grid is NULL");
    if (ifreq < 0 || ifreq >= G->n_freq) return fail(SOC_EINVAL, "ifreq out of range");
    if (n_packages < 0 || pkg_begin < 0 || pkg_count < 0 || pkg_begin + pkg_count > n_packages)
        return fail(SOC_EINVAL, "bad package range");
    if (!absorbed) return fail(SOC_EINVAL, "absorbed is NULL");
    if (!std::isfinite(weight)) return fail(SOC_EINVAL, "weight is not finite");
    if (flags & ~1u) return fail(SOC_EINVAL, "unknown flags");
    long long n_bg = 0;
    int rc = check_sources(G, src, n_packages, &n_bg);
    if (rc != SOC_OK) return rc;

    SimParams P;
    std::memset(&P, 0, sizeof(P));
    P.nx = G->nx; P.ny = G->ny; P.nz = G->nz; P.n_root = (int)G->n_root;
    P.cellw = G->d_cellw; P.parent = G->d_parent; P.n_total = (int)G->n_total; P.n_oct = (int)(G->n_octets > 0 ? G->n_octets : 1);
    P.kabs = G->kabs[ifreq]; P.ksca = G->ksca[ifreq]; P.g = G->g[ifreq];
    P.surf = 2.0 * ((double)G->ny * G->nz + (double)G->nz * G->nx + (double)G->nx * G->ny);
    P.n_bg = n_bg;
    if (src->beam) {
        P.is_beam = 1;
        for (int j = 0; j < 6; ++j) P.beam[j] = src->beam[j];
    } else {
        P.n_point = src->n_point;
        if (n_bg > 0) P.bg_e0 = kPi * src->bg_intensity * P.surf / (double)n_bg;
        const long long n_ps = n_packages - src->n_dust - n_bg;
        for (int k = 0; k < src->n_point; ++k) {
            for (int j = 0; j < 3; ++j) P.ps_pos[k][j] = src->ps_pos[3 * k + j];
            const long long count_k = n_ps / src->n_point + ((n_ps % src->n_point) > k ? 1 : 0);
            P.ps_e0[k] = count_k > 0 ? src->ps_lum[k] / (double)count_k : 0.0;
        }
    }
    // f1: dust re-emission -- the last n_dust ids; prefix sums of the counts, sum of the luminosities (synchronises)
    P.dust.n_const = n_packages;                 // no dust: every id is below n_const
    double dust_lum_total = 0.0;
    if (!src->beam && src->n_dust > 0 && pkg_count > 0) {
        rc = dust_prepare(G, ifreq, src, n_packages - src->n_dust, weight, &P.dust, &dust_lum_total, st);
        if (rc != SOC_OK) return rc;
    }
    P.pkg_begin = pkg_begin; P.pkg_end = pkg_begin + pkg_count;
    P.seed = seed; P.ifreq = ifreq; P.weight = weight;
    P.refill_threshold = G->opt_refill_threshold;
    P.absorbed = absorbed; P.replay = replay;
    P.counter = G->d_counters + slot; P.result = G->d_results + slot;

    SOC_CUDA(cudaMemsetAsync(G->d_counters + slot, 0, sizeof(unsigned long long), st));
    SOC_CUDA(cudaMemsetAsync(G->d_results + slot, 0, sizeof(DevResult), st));
    if (slot < (int)G->slot_group.size()) G->slot_group[slot] = 0;
    if (pkg_count == 0) return SOC_OK;
    const bool hier = G->n_levels > 1, f64 = (flags & SOC_GEOM_FP64) != 0, rep = replay != nullptr;
    if (G->opt_timing) {
        rc = ensure_events(G, slot + 1);
        if (rc != SOC_OK) return rc;
        SOC_CUDA(cudaEventRecord(G->ev0[slot], st));
        G->ev_after_photon = G->ev1[slot];
    }
    if (f64) {
        rc = hier ? (rep ? launch_photon<double, true, true>(G, P, st) : launch_photon<double, true, false>(G, P, st))
                  : (rep ? launch_photon<double, false, true>(G, P, st) : launch_photon<double, false, false>(G, P, st));
    } else {
        FastParams F;
        std::memset(&F, 0, sizeof(F));
        F.nx = G->nx; F.ny = G->ny; F.nz = G->nz; F.nbx = G->nbx; F.nby = G->nby;
        F.bsy = 8 * G->nbx; F.bsz = 8 * G->nbx * G->nby; F.nrp = G->nrp; F.n_root = (int)G->n_root;
        F.cellw = G->d_cellw_int; F.parent = G->d_parent_int;
        F.n_int = (int)G->n_int; F.n_oct = (int)(G->n_octets > 0 ? G->n_octets : 1); F.n_abi = (int)G->n_total;
        F.n_replay = (int)(pkg_count < (1ll << 31) ? pkg_count : (1ll << 31) - 1);
        F.kabs = (float)P.kabs; F.ksca = (float)P.ksca; F.g = (float)P.g;
        F.kratio = P.ksca > 0.0 ? (float)(P.kabs / P.ksca) : 0.0f;
        F.is_beam = P.is_beam; F.n_point = P.n_point; F.n_bg = P.n_bg; F.bg_e0 = P.bg_e0; F.surf = P.surf;
        std::memcpy(F.beam, P.beam, sizeof(F.beam));
        std::memcpy(F.ps_pos, P.ps_pos, sizeof(F.ps_pos));
        std::memcpy(F.ps_e0, P.ps_e0, sizeof(F.ps_e0));
        F.pkg_begin = P.pkg_begin; F.pkg_end = P.pkg_end; F.seed = P.seed; F.ifreq = P.ifreq;
        // service passes run with only the parked lanes active: where packages scatter many times (scattering depth of the
        // box >= 4) wait for 16 parked lanes instead of 8 (B200: -7 % on the UV launches of config 3, -2 % on config 5)
        {
            const int nm = G->nx > G->ny ? (G->nx > G->nz ? G->nx : G->nz) : (G->ny > G->nz ? G->ny : G->nz);
            F.service_threshold = G->opt_service_threshold > 0 ? G->opt_service_threshold
                                                               : (P.ksca * G->rho_mean * nm >= 4.0 ? 16 : 8);
        }
        const int auto_threshold = G->opt_service_threshold > 0 ? G->opt_service_threshold : 8;     // photon_q_kernel: 8 throughout
        // hot-cell cache: R = 3 (343 cells per source) while it fits in 40 KB per block, else R = 2; regular grids
        F.hot_r = -1;
        if (!hier && P.n_point > 0 && !P.is_beam && G->opt_hot_cache)
            F.hot_r = (size_t)P.n_point * 343 * sizeof(float) <= 40 * 1024 ? 3 : 2;
        F.acc = G->acc_sel ? G->d_acc_b : G->d_acc; F.replay = P.replay; F.counter = P.counter; F.result = P.result;
        // fp32 internal accumulator: deposits in units of the largest package energy of
        // this launch; falls back to the fp64 accumulator when a source class would underflow in those units
        double e_ref = P.is_beam ? 1.0 : P.bg_e0;
        for (int k = 0; k < P.n_point; ++k) e_ref = std::fmax(e_ref, P.ps_e0[k]);
        // dust packages carry L_c / n_c each: the mean package energy is the unit (the sums are fp32: any unit within
        // range will do; with weighted counts most packages carry about this much, capped cells more)
        F.dust = P.dust;
        if (P.dust.n_dust > 0) e_ref = std::fmax(e_ref, dust_lum_total / (double)P.dust.n_dust);
        F.e_ref = e_ref;
        bool acc32 = G->opt_acc32 != 0 && e_ref > 0.0 && std::isfinite(e_ref);
        if (acc32) {
            F.beam_rel = (float)(1.0 / e_ref);
            F.bg_rel = (float)(P.bg_e0 / e_ref);
            if (!P.is_beam && P.n_bg > 0 && P.bg_e0 > 0.0 && F.bg_rel < 1e-20f) acc32 = false;
            for (int k = 0; k < P.n_point; ++k) {
                F.ps_rel[k] = (float)(P.ps_e0[k] / e_ref);
                if (P.ps_e0[k] > 0.0 && F.ps_rel[k] < 1e-20f) acc32 = false;
            }
        }
        F.acc32 = G->acc_sel ? G->d_acc32_b : G->d_acc32;
        if (acc32 && F.hot_r >= 0) {
            double *&h = G->d_hot64[G->acc_sel];
            if (!h) {
                const size_t bytes = sizeof(double) * kHot64Len;
                SOC_CUDA(cudaMalloc(&h, bytes));
                SOC_CUDA(cudaMemsetAsync(h, 0, bytes, st));              // st = the stream that uses it
            }
            F.hot64 = h;
        }
        if (!acc32 && G->acc_sel && !G->d_acc_b) {           // fp64 fallback on the second stream: its own accumulator
            SOC_CUDA(big_malloc(&G->d_acc_b, sizeof(double) * (size_t)G->n_int));
            SOC_CUDA(cudaMemsetAsync(G->d_acc_b, 0, sizeof(double) * (size_t)G->n_int, st));   // st = the stream that uses it
            F.acc = G->d_acc_b;
        }
        const double w_eff = acc32 ? weight * e_ref : weight;
        // photon_q_kernel trades instructions for L2 requests: it wins where the working set (cell words + fp32
        // accumulator, 8 B per cell) does not stay in L2 (B200: 19.1 vs 20.2 ms per frequency on config 5) and loses
        // on L2-resident grids, which are bound by issue slots (3.2 vs 2.8 ms on config 3); profiles/README.md
        // and where packages do not scatter very often (every scattering parks the lane and reloads the half brick):
        // measured crossover on config 5, both kernels at their best occupancy, at a scattering depth of the box of 12-16
        const int n_max = G->nx > G->ny ? (G->nx > G->nz ? G->nx : G->nz) : (G->ny > G->nz ? G->ny : G->nz);
        const bool big = 8ll * G->n_int > l2_share(G, 64) && P.ksca * G->rho_mean * n_max < 12.0;
        const bool v2 = !hier && acc32 && (G->opt_kernel == 2 || (G->opt_kernel == 0 && big)) && pkg_count < (1ll << 32);
        if (v2) F.service_threshold = auto_threshold;
        // z-slab blocking: the cell words and the accumulator of one slab stay in L2 while it is served.
        // Two slabs of 70 MB serve config 5 on B200 (126 MB of L2) as well as four or eight do (same hit rate, 3 GB of DRAM
        // traffic per frequency against 54 GB) with the fewest suspensions; where packages scatter so often that the walk
        // is bound by the service passes (scattering depth of the box >= 12) photon_fast_kernel without slabs is faster
        int n_slabs = G->opt_slabs;
        if (n_slabs == 0) n_slabs = 8ll * G->n_int > l2_share(G, 96) ? (int)((8ll * G->n_int + l2_share(G, 80) - 1) / l2_share(G, 80)) : 1;
        if (n_slabs > G->nbz / 2) n_slabs = G->nbz / 2;
        if (n_slabs > kMaxSlabs) n_slabs = kMaxSlabs;
        const bool slab = !hier && acc32 && !rep && n_slabs >= 2 &&
                          (G->opt_kernel == 2 || (G->opt_kernel == 0 && P.ksca * G->rho_mean * n_max < 12.0));
        if (slab) {
            // one sweep up, one down; what scatters back across a slab boundary after that is left to the last, whole-grid
            // phase (more sweeps were slower at every scattering depth)
            const int sweeps = G->opt_slab_sweeps > 0 ? G->opt_slab_sweeps : 2;
            F.service_threshold = auto_threshold;
            // a queued state carries its package index in 24 bits: at most 2^24 packages per sequence of phases
            const long long chunk = G->opt_slab_chunk > 0 ? G->opt_slab_chunk : (1ll << 24);
            rc = SOC_OK;
            for (long long b = P.pkg_begin; b < P.pkg_end && rc == SOC_OK; b += chunk) {
                F.pkg_begin = b; F.pkg_end = b + chunk < P.pkg_end ? b + chunk : P.pkg_end;
                const bool last = F.pkg_end == P.pkg_end;
                if (F.dust.n_dust > 0)
                    rc = G->opt_stats ? launch_slab<true, true>(G, F, n_slabs, sweeps, w_eff, absorbed, last, st)
                                      : launch_slab<false, true>(G, F, n_slabs, sweeps, w_eff, absorbed, last, st);
                else
                    rc = G->opt_stats ? launch_slab<true, false>(G, F, n_slabs, sweeps, w_eff, absorbed, last, st)
                                      : launch_slab<false, false>(G, F, n_slabs, sweeps, w_eff, absorbed, last, st);
            }
        } else {
        const int sel = (v2 ? 8 : 0) | (hier ? 4 : 0) | ((rep || G->opt_stats) ? 2 : 0) | (acc32 ? 1 : 0);
#define SOC_LF(H, R, A, Q) (F.dust.n_dust > 0 ? launch_fast<H, R, A, Q, true>(G, F, w_eff, absorbed, st) \
                                              : launch_fast<H, R, A, Q, false>(G, F, w_eff, absorbed, st))
        switch (sel) {
        case 9: rc = SOC_LF(false, false, true, true); break;
        case 11: rc = SOC_LF(false, true, true, true); break;
        case 0: rc = SOC_LF(false, false, false, false); break;
        case 1: rc = SOC_LF(false, false, true, false); break;
        case 2: rc = SOC_LF(false, true, false, false); break;
        case 3: rc = SOC_LF(false, true, true, false); break;
        case 4: rc = SOC_LF(true, false, false, false); break;
        case 5: rc = SOC_LF(true, false, true, false); break;
        case 6: rc = SOC_LF(true, true, false, false); break;
        default: rc = SOC_LF(true, true, true, false); break;
        }
#undef SOC_LF
        }
    }
    if (rc == SOC_OK && G->opt_timing) {
        if (G->ev_after_photon) SOC_CUDA(cudaEventRecord(G->ev1[slot], st));
        G->ev_set[slot] = 1;
    }
    G->ev_after_photon = nullptr;
    return rc;
}

// Frequencies [f0, f0 + J) in ONE launch (FastParams::job): returns SOC_OK, an error, or 1 = "not eligible, launch them
// one by one" (sources that differ in more than their energies, dust or beam packages, a grid served by photon_q_kernel
// or by the hot-cell cache, energies that would underflow the common fp32 unit).
int enqueue_group(soc_grid *G, int f0, int J, const soc_sources *src, long long n_packages, unsigned long long seed,
                  const double *w, long long pkg_begin, long long pkg_count, double *absorbed, int slot0, cudaStream_t st)
{
    const bool hier = G->n_levels > 1;
    if (J < 1 || J > kMaxJobs || !G->opt_acc32 || pkg_count <= 0 || !absorbed) return 1;
    if (n_packages < 0 || pkg_begin < 0 || pkg_begin + pkg_count > n_packages) return 1;
    if (!hier && (8ll * G->n_int > l2_share(G, 64) || G->opt_kernel == 2)) return 1;
    long long n_bg0 = 0;
    for (int j = 0; j < J; ++j) {
        long long n_bg = 0;
        const int rc = check_sources(G, src + j, n_packages, &n_bg);
        if (rc != SOC_OK) return rc;
        if (src[j].beam || src[j].n_dust > 0 || !std::isfinite(w[j])) return 1;
        if (j == 0) { n_bg0 = n_bg; continue; }
        if (n_bg != n_bg0 || src[j].n_point != src[0].n_point) return 1;
        for (int k = 0; k < 3 * src[0].n_point; ++k)
            if (src[j].ps_pos[k] != src[0].ps_pos[k]) return 1;
    }
    FastParams F;
    std::memset(&F, 0, sizeof(F));
    F.nx = G->nx; F.ny = G->ny; F.nz = G->nz; F.nbx = G->nbx; F.nby = G->nby;
    F.bsy = 8 * G->nbx; F.bsz = 8 * G->nbx * G->nby; F.nrp = G->nrp; F.n_root = (int)G->n_root;
    F.cellw = G->d_cellw_int; F.parent = G->d_parent_int;
    F.n_int = (int)G->n_int; F.n_oct = (int)(G->n_octets > 0 ? G->n_octets : 1); F.n_abi = (int)G->n_total; F.n_replay = 1;
    F.surf = 2.0 * ((double)G->ny * G->nz + (double)G->nz * G->nx + (double)G->nx * G->ny);
    F.n_point = src[0].n_point; F.n_bg = n_bg0;
    for (int k = 0; k < F.n_point; ++k)
        for (int a = 0; a < 3; ++a) F.ps_pos[k][a] = src[0].ps_pos[3 * k + a];
    F.dust.n_const = n_packages;
    F.seed = seed; F.ifreq = f0;
    F.hot_r = -1;
    if (!hier && F.n_point > 0 && G->opt_hot_cache) F.hot_r = (size_t)F.n_point * 343 * sizeof(float) <= 40 * 1024 ? 3 : 2;
    F.n_jobs = J; F.job_pkgs = pkg_count; F.pkg_begin = pkg_begin; F.pkg_end = pkg_begin + (long long)J * pkg_count;
    const int nm = G->nx > G->ny ? (G->nx > G->nz ? G->nx : G->nz) : (G->ny > G->nz ? G->ny : G->nz);
    const long long n_ps = n_packages - n_bg0;
    double e_ref = 0.0, depth = 0.0;
    std::vector<double> bg_e0((size_t)J, 0.0);
    for (int j = 0; j < J; ++j) {
        JobParams &Q = F.job[j];
        const double kabs = G->kabs[f0 + j], ksca = G->ksca[f0 + j];
        Q.kabs = (float)kabs; Q.ksca = (float)ksca; Q.g = (float)G->g[f0 + j];
        Q.kratio = ksca > 0.0 ? (float)(kabs / ksca) : 0.0f;
        Q.ifreq = f0 + j;
        depth = std::fmax(depth, ksca * G->rho_mean * nm);
        if (n_bg0 > 0) Q.bg_e0 = kPi * src[j].bg_intensity * F.surf / (double)n_bg0;
        e_ref = std::fmax(e_ref, w[j] * Q.bg_e0);
        for (int k = 0; k < F.n_point; ++k) {
            const long long count_k = n_ps / F.n_point + ((n_ps % F.n_point) > k ? 1 : 0);
            Q.ps_e0[k] = count_k > 0 ? src[j].ps_lum[k] / (double)count_k : 0.0;
            e_ref = std::fmax(e_ref, w[j] * Q.ps_e0[k]);
        }
    }
    if (!(e_ref > 0.0) || !std::isfinite(e_ref)) return 1;
    for (int j = 0; j < J; ++j) {
        JobParams &Q = F.job[j];
        Q.bg_rel = (float)(w[j] * Q.bg_e0 / e_ref);
        if (n_bg0 > 0 && Q.bg_e0 > 0.0 && !(Q.bg_rel >= 1e-20f)) return 1;
        for (int k = 0; k < F.n_point; ++k) {
            Q.ps_rel[k] = (float)(w[j] * Q.ps_e0[k] / e_ref);
            if (Q.ps_e0[k] > 0.0 && !(Q.ps_rel[k] >= 1e-20f)) return 1;
        }
    }
    // the jobs share one fp32 accumulator: a frequency whose packages carry much less than the launch's unit loses its
    // deposits wherever a brighter one dominates the sum (they fall below half the last bit), one-sidedly: measured on the
    // smoke problem (three frequencies decades apart, point sources in an octree) as 1e-6 of the absorbed energy.  Such a
    // frequency is launched on its own (the caller retries the group from the next frequency): below 1e-2 of the unit where
    // point sources make cells that collect 1e4 and more deposits per launch; below 1e-7 with the background alone, where a
    // cell collects some tens per launch and what such a frequency can lose is 1e-7 of the launch's energy at most
    // (config 4' with its faintest UV frequencies grouped: cells against counters 9e-9)
    for (int j = 0; j < J; ++j) {
        float top = F.job[j].bg_rel;
        for (int k = 0; k < F.n_point; ++k) top = std::fmax(top, F.job[j].ps_rel[k]);
        if (!(top >= (F.n_point > 0 ? 1e-2f : kGroupMinRel))) return 1;
        // (and with the group size chosen by the library, point sources keep one frequency per launch altogether: config 3
        //  in fours gains 3 % and holds its cells to 6e-7 of the counters instead of 3e-8)
        if (J > 1 && F.n_point > 0 && G->opt_group == 0) return 1;
    }
    F.e_ref = e_ref;
    F.service_threshold = G->opt_service_threshold > 0 ? G->opt_service_threshold : (depth >= 4.0 ? 16 : 8);
    F.acc = G->acc_sel ? G->d_acc_b : G->d_acc; F.acc32 = G->acc_sel ? G->d_acc32_b : G->d_acc32;
    if (F.hot_r >= 0) {
        double *&h = G->d_hot64[G->acc_sel];
        if (!h) {
            const size_t bytes = sizeof(double) * kHot64Len;
            SOC_CUDA(cudaMalloc(&h, bytes));
            SOC_CUDA(cudaMemsetAsync(h, 0, bytes, st));                  // st = the stream that uses it
        }
        F.hot64 = h;
    }
    F.counter = G->d_counters + slot0; F.result = G->d_results + slot0;
    SOC_CUDA(cudaMemsetAsync(G->d_counters + slot0, 0, sizeof(unsigned long long) * (size_t)J, st));
    SOC_CUDA(cudaMemsetAsync(G->d_results + slot0, 0, sizeof(DevResult) * (size_t)J, st));
    if ((int)G->slot_group.size() < slot0 + J) G->slot_group.resize((size_t)(slot0 + J), 0);
    for (int j = 0; j < J; ++j) G->slot_group[slot0 + j] = j == 0 ? J : 0;
    if (G->opt_timing) {
        const int rc = ensure_events(G, slot0 + J);
        if (rc != SOC_OK) return rc;
        SOC_CUDA(cudaEventRecord(G->ev0[slot0], st));
        G->ev_after_photon = G->ev1[slot0];
    }
    int rc;
    if (hier) rc = G->opt_stats ? launch_fast<true, true, true, false, false, true>(G, F, e_ref, absorbed, st)
                                : launch_fast<true, false, true, false, false, true>(G, F, e_ref, absorbed, st);
    else rc = G->opt_stats ? launch_fast<false, true, true, false, false, true>(G, F, e_ref, absorbed, st)
                           : launch_fast<false, false, true, false, false, true>(G, F, e_ref, absorbed, st);
    if (rc == SOC_OK && G->opt_timing) {
        // every member of the group carries the group's event pair: soc_get_timings divides the time among them
        for (int j = 0; j < J; ++j) G->ev_set[slot0 + j] = 1;
        for (int j = 1; j < J; ++j) {
            SOC_CUDA(cudaEventRecord(G->ev0[slot0 + j], st));
            SOC_CUDA(cudaEventRecord(G->ev1[slot0 + j], st));
        }
    }
    G->ev_after_photon = nullptr;
    return rc;
}

int fetch_results(soc_grid *G, int n, soc_freq_result *out, cudaStream_t st)
{
    SOC_CUDA(cudaMemcpyAsync(G->h_results, G->d_results, sizeof(DevResult) * n, cudaMemcpyDeviceToHost, st));
    SOC_CUDA(cudaStreamSynchronize(st));
    for (int i = 0; i < n; ++i) {
        out[i].emitted = G->h_results[i].emitted; out[i].escaped = G->h_results[i].escaped;
        out[i].absorbed = G->h_results[i].absorbed; out[i].cell_steps = G->h_results[i].cell_steps;
        out[i].scatterings = G->h_results[i].scatterings; out[i].terminated = G->h_results[i].terminated;
        float drift;
        std::memcpy(&drift, &G->h_results[i].drift_bits, sizeof(float));
        out[i].weight_drift = (double)drift;
        out[i].gather_requests = G->h_results[i].gathers; out[i].red_requests = G->h_results[i].reds;
        out[i].suspensions = G->h_results[i].suspensions; out[i].queue_refusals = G->h_results[i].refusals;
    }
    return SOC_OK;
}

void trapezoid(const std::vector<double> &nu, std::vector<double> &w)
{
    const size_t n = nu.size();
    w.assign(n, 1.0);
    if (n < 2) return;
    for (size_t i = 0; i < n; ++i) {
        const double lo = nu[i > 0 ? i - 1 : 0], hi = nu[i + 1 < n ? i + 1 : n - 1];
        w[i] = 0.5 * (hi - lo);
    }
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// Scratch of soc_update_temperatures_ali_static, the ALI temperature update for callers that must not allocate device
// memory (soc.h says who they are).  The regular call keeps its per-cell work array (the effective absorbed energy
// (A - S) / (1 - beta)) in a buffer it allocates on first use and stages the temperature table through pinned memory it
// allocates too.  Here both live in this one array, which is part of the library image: every GPU that loads the
// library holds its 16 MiB + 32 KiB from the moment the module is loaded until the process ends, whether or not the
// entry point is ever called.
//   [0, kStaticMaxCells)                 effective absorbed energy per cell
//   [kStaticMaxCells, end)               the temperature table (up to kStaticMaxTable floats)
// In host code the NAME g_static_scratch is only the host-side handle of the symbol, not an address the GPU can use:
// the device address is looked up once per device by static_scratch() below and that pointer is what kernels receive.
// ------------------------------------------------------------------------------------------------
constexpr long long kStaticMaxCells = 1ll << 21;            // 2 097 152 cells: a 128^3 regular grid (config 3) fits exactly
constexpr int kStaticMaxTable = 8192;                       // floats; the same cap as soc_update_temperatures
static __device__ __align__(256) double g_static_scratch[kStaticMaxCells + kStaticMaxTable / 2];

namespace {

constexpr int kStaticMaxDevices = 64;
double *g_static_ptr[kStaticMaxDevices];                    // device address of g_static_scratch on device i, once known
std::mutex g_static_mutex;

// Device address of the scratch array on `device`, which must be the current device.  The first call per device asks
// the runtime for it (this is the set-up; it allocates nothing, the array came with the module) and keeps the answer.
int static_scratch(int device, double **out)
{
    if (device < 0 || device >= kStaticMaxDevices) return fail(SOC_EINVAL, "soc_update_temperatures_ali_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[device]) {
        double *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_static_scratch);
        if (e != cudaSuccess || !p)
            return fail(SOC_ECUDA, std::string("soc_update_temperatures_ali_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        g_static_ptr[device] = p;
    }
    *out = g_static_ptr[device];
    return SOC_OK;
}

}  // namespace

extern "C" {

const char *soc_last_error(void) { return g_last_error.c_str(); }
const char *soc_version(void) { return "soc_b200 0.1 (sm_100a)"; }
uint64_t soc_launch_count(void) { return g_launches; }

}  // extern "C"

namespace {
int64_t release_caches()
{
    int64_t bytes = 0;
    std::lock_guard<std::mutex> lock(g_queue_cache_mutex);
    if (!g_queue_cache.empty()) cudaDeviceSynchronize();
    for (const CachedBuffer &b : g_queue_cache) {
        cudaFree(b.ptr);
        bytes += (int64_t)(b.entries * kQueueEntryBytes);
    }
    g_queue_cache.clear();
    std::lock_guard<std::mutex> lock2(g_big_mutex);
    if (!g_big_cache.empty()) cudaDeviceSynchronize();
    for (const BigBuffer &b : g_big_cache) { cudaFree(b.ptr); bytes += (int64_t)b.bytes; }
    g_big_cache.clear();
    return bytes;
}
}  // namespace

extern "C" {

int64_t soc_release_cached_memory(void) { return release_caches(); }

int64_t soc_checked_violations(void)
{
#ifdef SOC_CHECKED
    unsigned int v = 0;
    if (cudaDeviceSynchronize() != cudaSuccess) return -2;
    if (cudaMemcpyFromSymbol(&v, g_violations, sizeof(v)) != cudaSuccess) return -2;
    return (int64_t)v;
#else
    return -1;
#endif
}

void soc_grid_destroy(soc_grid *G)
{
    if (!G) return;
    cudaDeviceSynchronize();                     // (the cached buffers may be handed to another grid at once)
    big_free(G->d_cellw); big_free(G->d_parent); cudaFree(G->d_results); cudaFree(G->d_counters);
    cudaFree(G->d_table); big_free(G->d_cellw_int); big_free(G->d_parent_int); big_free(G->d_acc); big_free(G->d_acc32);
    if (G->h_results) cudaFreeHost(G->h_results);
    if (G->h_table) cudaFreeHost(G->h_table);
    if (G->h_scalars) cudaFreeHost(G->h_scalars);
    cudaFree(G->d_dust_first); cudaFree(G->d_scan_blocks); cudaFree(G->d_scalars); cudaFree(G->d_freqtab); big_free(G->d_eff);
    if (G->ev_table) cudaEventDestroy(G->ev_table);
    big_free(G->d_acc32_b); big_free(G->d_acc_b);
    for (int i = 0; i < 2; ++i) {
        if (G->d_slab_q[i]) {                    // the queue buffers go to the process-wide cache (soc.h); the smallest is evicted
            cudaDeviceSynchronize();
            std::lock_guard<std::mutex> lock(g_queue_cache_mutex);
            g_queue_cache.push_back({G->d_slab_q[i], G->slab_q_entries[i], G->device});
            if (g_queue_cache.size() > kQueueCacheMax) {
                size_t small = 0;
                for (size_t k = 1; k < g_queue_cache.size(); ++k)
                    if (g_queue_cache[k].entries < g_queue_cache[small].entries) small = k;
                cudaFree(g_queue_cache[small].ptr);
                g_queue_cache.erase(g_queue_cache.begin() + small);
            }
        }
        cudaFree(G->d_slab_cnt[i]); cudaFree(G->d_hot64[i]);
    }
    if (G->aux) cudaStreamDestroy(G->aux);
    if (G->ev_fork) cudaEventDestroy(G->ev_fork);
    if (G->ev_join) cudaEventDestroy(G->ev_join);
    if (G->ev_unpad[0]) cudaEventDestroy(G->ev_unpad[0]);
    if (G->ev_unpad[1]) cudaEventDestroy(G->ev_unpad[1]);
    for (cudaEvent_t e : G->ev0) cudaEventDestroy(e);
    for (cudaEvent_t e : G->ev1) cudaEventDestroy(e);
    delete G;
}

int64_t soc_grid_n_total(const soc_grid *G) { return G ? G->n_total : 0; }

int soc_grid_create(const soc_grid_desc *d, soc_grid **out)
{
    if (!d || !out) return fail(SOC_EINVAL, "NULL argument");
    *out = nullptr;
    if (d->nx < 1 || d->ny < 1 || d->nz < 1) return fail(SOC_EINVAL, "root grid dimensions must be >= 1");
    if (d->n_levels < 1 || d->n_levels > SOC_MAX_LEVELS) return fail(SOC_EINVAL, "n_levels out of range");
    if (!d->n_cells || !d->density) return fail(SOC_EINVAL, "n_cells / density is NULL");
    if (d->n_levels > 1 && !d->child) return fail(SOC_EINVAL, "child is NULL for a hierarchical grid");
    if (d->n_freq < 1 || !d->freq_hz || !d->kabs || !d->ksca || !d->g) return fail(SOC_EINVAL, "dust tables missing");
    if (d->n_cells[0] != (int64_t)d->nx * d->ny * d->nz) return fail(SOC_EINVAL, "n_cells[0] != nx*ny*nz");
    soc_grid *G = new (std::nothrow) soc_grid;
    if (!G) return fail(SOC_ENOMEM, "out of host memory");
    struct Guard { soc_grid *g; ~Guard() { if (g) soc_grid_destroy(g); } } guard{G};
    G->nx = d->nx; G->ny = d->ny; G->nz = d->nz; G->n_levels = d->n_levels; G->n_freq = d->n_freq;
    for (int l = 0; l < d->n_levels; ++l) {
        if (d->n_cells[l] < 0 || (l > 0 && d->n_cells[l] % 8 != 0)) return fail(SOC_EINVAL, "level sizes must be multiples of 8");
        G->level_off[l + 1] = G->level_off[l] + d->n_cells[l];
    }
    G->n_total = G->level_off[d->n_levels];
    G->n_root = d->n_cells[0];
    if (G->n_total >= (1ll << 31)) return fail(SOC_EINVAL, "more than 2^31 cells");
    G->n_octets = (G->n_total - G->n_root) / 8;
    for (int f = 0; f < d->n_freq; ++f) {
        if (!std::isfinite(d->freq_hz[f]) || !(d->freq_hz[f] > 0) || (f > 0 && !(d->freq_hz[f] > d->freq_hz[f - 1])))
            return fail(SOC_EINVAL, "freq_hz must be positive and strictly ascending");
        if (!(d->kabs[f] >= 0) || !(d->ksca[f] >= 0) || !std::isfinite(d->kabs[f]) || !std::isfinite(d->ksca[f]))
            return fail(SOC_EINVAL, "kabs / ksca must be finite and >= 0");
        if (!(std::fabs(d->g[f]) < 1.0)) return fail(SOC_EINVAL, "|g| must be < 1");
    }
    G->freq.assign(d->freq_hz, d->freq_hz + d->n_freq);
    G->kabs.assign(d->kabs, d->kabs + d->n_freq);
    G->ksca.assign(d->ksca, d->ksca + d->n_freq);
    G->g.assign(d->g, d->g + d->n_freq);

    // cell words and reverse links (the link replaces the density of the parent; one reverse
    // link per octet)
    std::vector<uint32_t> cellw;
    std::vector<int32_t> parent;
    // grids of >= 2^20 cells are converted and validated on the GPU: regular grids by leafwords_kernel, hierarchies by
    // hierwords_kernel + parent_internal_kernel (the host loops below cost 40 ms for the 11 M cells of config 4')
    const bool big = G->n_total >= (1ll << 20);
    const bool words_done = big;
    const bool hier_gpu = big && d->child != nullptr;
    const size_t n_par = (size_t)(G->n_octets > 0 ? G->n_octets : 1);
    try {
        if (!big) { cellw.resize((size_t)G->n_total); parent.assign(n_par, INT32_MIN); }
    } catch (const std::bad_alloc &) {
        return fail(SOC_ENOMEM, "out of host memory");
    }
    for (int l = 0; l < d->n_levels && !words_done; ++l) {
        for (long long c = 0; c < d->n_cells[l]; ++c) {
            const long long gid = G->level_off[l] + c;
            const int32_t ch = d->child ? d->child[gid] : -1;
            if (ch < 0) {
                const float r = d->density[gid];
                if (!(r >= 0.0f) || !std::isfinite(r)) return fail(SOC_EINVAL, "leaf density must be finite and >= 0");
                float rp = r + 0.0f;                         // -0.0 -> +0.0 so that the sign bit means "parent"
                uint32_t bits;
                std::memcpy(&bits, &rp, 4);
                cellw[(size_t)gid] = bits & 0x7fffffffu;
                continue;
            }
            if (l + 1 >= d->n_levels || (ch & 7) != 0 || (long long)ch + 8 > d->n_cells[l + 1])
                return fail(SOC_EINVAL, "child index out of range or not a multiple of 8");
            const long long child_rel = G->level_off[l + 1] + ch - G->n_root;
            if (parent[(size_t)(child_rel >> 3)] != INT32_MIN) return fail(SOC_EINVAL, "octet has two parents");
            parent[(size_t)(child_rel >> 3)] = (int32_t)(gid - G->n_root);
            cellw[(size_t)gid] = 0x80000000u | (uint32_t)child_rel;
        }
    }
    for (long long o = 0; o < G->n_octets && !words_done; ++o)
        if (parent[(size_t)o] == INT32_MIN) return fail(SOC_EINVAL, "octet without a parent");
    if (!words_done) {
        double sum = 0.0;
        long long cnt = 0;
        for (long long c = 0; c < G->n_root; ++c)
            if ((int32_t)cellw[(size_t)c] >= 0) { sum += (double)d->density[c]; cnt += 1; }
        G->rho_mean = cnt > 0 ? sum / (double)cnt : 0.0;
    }

    SOC_CUDA(cudaGetDevice(&G->device));
    SOC_CUDA(cudaDeviceGetAttribute(&G->n_sm, cudaDevAttrMultiProcessorCount, G->device));
    {
        int l2 = 0;
        SOC_CUDA(cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, G->device));
        if (l2 > 0) G->l2_bytes = l2;
    }
    SOC_CUDA(big_malloc(&G->d_cellw, sizeof(uint32_t) * (size_t)G->n_total));
    SOC_CUDA(big_malloc(&G->d_parent, sizeof(int32_t) * n_par));
    SOC_CUDA(cudaMalloc(&G->d_table, sizeof(float) * 8192));
    if (hier_gpu) {
        double *d_sum = nullptr;
        int32_t *d_child = nullptr;
        struct Tmp { double *&a; int32_t *&b; ~Tmp() { cudaFree(a); big_free(b); } } tmp{d_sum, d_child};
        SOC_CUDA(cudaMalloc(&d_sum, 32));
        SOC_CUDA(cudaMemset(d_sum, 0, 32));
        SOC_CUDA(big_malloc(&d_child, sizeof(int32_t) * (size_t)G->n_total));
        SOC_CUDA(cudaMemcpy(G->d_cellw, d->density, sizeof(float) * (size_t)G->n_total, cudaMemcpyHostToDevice));
        SOC_CUDA(cudaMemcpy(d_child, d->child, sizeof(int32_t) * (size_t)G->n_total, cudaMemcpyHostToDevice));
        HierParams H;
        std::memset(&H, 0, sizeof(H));
        H.cellw = G->d_cellw; H.child = d_child; H.parent = G->d_parent; H.n_total = G->n_total; H.n_root = G->n_root;
        H.n_levels = G->n_levels;
        for (int l = 0; l <= G->n_levels; ++l) H.level_off[l] = G->level_off[l];
        H.sum_out = d_sum; H.flags = reinterpret_cast<int *>(d_sum + 2);
        fill_i32_kernel<<<G->n_sm * 4, 256>>>(G->d_parent, (long long)n_par, INT32_MIN);
        hierwords_kernel<<<G->n_sm * 8, 256>>>(H);
        g_launches += 2;
        double h_sum[4] = {0.0, 0.0, 0.0, 0.0};
        SOC_CUDA(cudaMemcpy(h_sum, d_sum, 32, cudaMemcpyDeviceToHost));
        int bad = 0;
        std::memcpy(&bad, &h_sum[2], sizeof(int));
        if (bad & 1) return fail(SOC_EINVAL, "leaf density must be finite and >= 0");
        if (bad & 2) return fail(SOC_EINVAL, "child index out of range or not a multiple of 8");
        if (bad & 4) return fail(SOC_EINVAL, "octet has two parents");
        G->rho_mean = h_sum[1] > 0.0 ? h_sum[0] / h_sum[1] : 0.0;
    } else if (words_done) {
        double *d_sum = nullptr;
        SOC_CUDA(cudaMalloc(&d_sum, 16));
        SOC_CUDA(cudaMemset(d_sum, 0, 16));
        SOC_CUDA(cudaMemcpy(G->d_cellw, d->density, sizeof(float) * (size_t)G->n_total, cudaMemcpyHostToDevice));
        leafwords_kernel<<<G->n_sm * 8, 256>>>(G->d_cellw, G->n_total, d_sum, reinterpret_cast<int *>(d_sum + 1));
        g_launches += 1;
        double h_sum[2] = {0.0, 0.0};
        cudaError_t e = cudaMemcpy(h_sum, d_sum, 16, cudaMemcpyDeviceToHost);
        cudaFree(d_sum);
        if (e != cudaSuccess) return fail(SOC_ECUDA, std::string("leafwords_kernel: ") + cudaGetErrorString(e));
        int bad = 0;
        std::memcpy(&bad, &h_sum[1], sizeof(int));
        if (bad) return fail(SOC_EINVAL, "leaf density must be finite and >= 0");
        G->rho_mean = h_sum[0] / (double)G->n_total;
    } else {
        SOC_CUDA(cudaMemcpy(G->d_cellw, cellw.data(), sizeof(uint32_t) * (size_t)G->n_total, cudaMemcpyHostToDevice));
    }
    if (!big) SOC_CUDA(cudaMemcpy(G->d_parent, parent.data(), sizeof(int32_t) * n_par, cudaMemcpyHostToDevice));
    else if (!hier_gpu) SOC_CUDA(cudaMemset(G->d_parent, 0, sizeof(int32_t) * n_par));
    // internal layout: root grid in 2x2x2 bricks with ghost cells around it (they hold the sentinel; cell ix
    // sits at X = ix + 2, so the low side has a whole ghost brick and the high side at least one ghost cell),
    // octet levels shifted behind it
    {
        const long long nbx = ((long long)G->nx + 4) / 2, nby = ((long long)G->ny + 4) / 2, nbz = ((long long)G->nz + 4) / 2;
        const long long nrp = 8 * nbx * nby * nbz;
        const long long n_int = nrp + (G->n_total - G->n_root);
        if (n_int >= (1ll << 31)) return fail(SOC_EINVAL, "more than 2^31 cells in the padded layout");
        G->nbx = (int)nbx; G->nby = (int)nby; G->nbz = (int)nbz; G->nrp = (int)nrp; G->n_int = n_int;
        std::vector<int32_t> pi;
        try {
            if (!big) pi.assign(n_par, 0);
        } catch (const std::bad_alloc &) {
            return fail(SOC_ENOMEM, "out of host memory");
        }
        auto internal = [&](long long gid) -> long long {
            if (gid >= G->n_root) return nrp + (gid - G->n_root);
            const long long ix = gid % G->nx, r = gid / G->nx, iy = r % G->ny, iz = r / G->ny;
            const long long X = ix + 2, Y = iy + 2, Z = iz + 2;
            return 8 * ((X >> 1) + nbx * ((Y >> 1) + nby * (Z >> 1))) + (X & 1) + 2 * (Y & 1) + 4 * (Z & 1);
        };
        for (long long o = 0; o < G->n_octets && !big; ++o) pi[(size_t)o] = (int32_t)internal((long long)parent[(size_t)o] + G->n_root);
        SOC_CUDA(big_malloc(&G->d_cellw_int, sizeof(uint32_t) * (size_t)n_int));
        SOC_CUDA(big_malloc(&G->d_parent_int, sizeof(int32_t) * n_par));
        SOC_CUDA(big_malloc(&G->d_acc, sizeof(double) * (size_t)n_int));
        repad_kernel<<<G->n_sm * 8, 256>>>(G->d_cellw, G->d_cellw_int, G->nx, G->ny, G->nz, (int)nbx, (int)nby, nrp, G->n_root, n_int);
        g_launches += 1;
        SOC_CUDA(cudaGetLastError());
        if (!big) SOC_CUDA(cudaMemcpy(G->d_parent_int, pi.data(), sizeof(int32_t) * n_par, cudaMemcpyHostToDevice));
        else if (hier_gpu) {
            int *d_f = nullptr;
            SOC_CUDA(cudaMalloc(&d_f, 4));
            SOC_CUDA(cudaMemset(d_f, 0, 4));
            parent_internal_kernel<<<G->n_sm * 4, 256>>>(G->d_parent, G->d_parent_int, G->n_octets, G->nx, G->ny, nbx, nby, nrp, G->n_root, d_f);
            g_launches += 1;
            int f = 0;
            cudaError_t e = cudaMemcpy(&f, d_f, 4, cudaMemcpyDeviceToHost);
            cudaFree(d_f);
            if (e != cudaSuccess) return fail(SOC_ECUDA, cudaGetErrorString(e));
            if (f & 8) return fail(SOC_EINVAL, "octet without a parent");
        } else SOC_CUDA(cudaMemset(G->d_parent_int, 0, sizeof(int32_t) * n_par));
        SOC_CUDA(cudaMemset(G->d_acc, 0, sizeof(double) * (size_t)n_int));
        SOC_CUDA(big_malloc(&G->d_acc32, sizeof(float) * (size_t)n_int));
        SOC_CUDA(cudaMemset(G->d_acc32, 0, sizeof(float) * (size_t)n_int));
    }
    int rc = ensure_slots(G, d->n_freq > 8 ? d->n_freq : 8);
    if (rc != SOC_OK) return rc;
    // the conversion kernels and memsets above ran on the legacy stream: a caller's non-blocking stream is not ordered
    // after it, so the grid is complete before the call returns
    SOC_CUDA(cudaDeviceSynchronize());
    guard.g = nullptr;
    *out = G;
    return SOC_OK;
}

int soc_freq_weights(const soc_grid *G, double *w)
{
    if (!G || !w) return fail(SOC_EINVAL, "NULL argument");
    std::vector<double> ww;
    trapezoid(G->freq, ww);
    for (int f = 0; f < G->n_freq; ++f) w[f] = ww[f];
    return SOC_OK;
}

int soc_set_option(soc_grid *G, const char *key, int64_t value)
{
    if (!G || !key) return fail(SOC_EINVAL, "NULL argument");
    const std::string k(key);
    if (k == "blocks_per_sm" && value >= 0 && value <= 32) G->opt_blocks_per_sm = (int)value;
    else if (k == "threads" && (value == 64 || value == 128 || value == 192 || value == 256)) G->opt_threads = (int)value;
    else if (k == "refill_threshold" && value >= 1 && value <= 32) G->opt_refill_threshold = (int)value;
    else if (k == "service_threshold" && value >= 0 && value <= 32) G->opt_service_threshold = (int)value;
    else if (k == "timing" && (value == 0 || value == 1)) G->opt_timing = (int)value;
    else if (k == "hot_cache" && (value == 0 || value == 1)) G->opt_hot_cache = (int)value;
    else if (k == "stats" && (value == 0 || value == 1)) G->opt_stats = (int)value;
    else if (k == "kernel" && value >= 0 && value <= 2) G->opt_kernel = (int)value;
    else if (k == "slabs" && value >= 0 && value <= 62) G->opt_slabs = (int)value;
    else if (k == "slab_sweeps" && value >= 0 && value <= 64) G->opt_slab_sweeps = (int)value;
    else if (k == "slab_queue_limit" && value >= 0 && value < (1ll << 32)) G->opt_slab_queue_limit = value;
    else if (k == "slab_chunk" && value >= 0 && value <= (1ll << 24)) G->opt_slab_chunk = value;
    else if (k == "group" && value >= 0 && value <= kMaxJobs) G->opt_group = (int)value;
    else if (k == "overlap" && (value == 0 || value == 1)) G->opt_overlap = (int)value;
    else if (k == "carveout" && value >= -1 && value <= 100) G->opt_carveout = (int)value;
    else if (k == "acc32" && (value == 0 || value == 1)) G->opt_acc32 = (int)value;
    else return fail(SOC_EINVAL, "unknown option or value out of range: " + k);
    return SOC_OK;
}

int soc_get_timings(soc_grid *G, int32_t n, float *ms)
{
    if (!G || !ms || n < 0) return fail(SOC_EINVAL, "bad argument");
    for (int i = 0; i < n; ++i) {
        ms[i] = -1.0f;
        if (i < (int)G->ev_set.size() && G->ev_set[i]) {
            SOC_CUDA(cudaEventSynchronize(G->ev1[i]));
            if (G->last_overlap && i > 0 && G->ev_set[i - 1]) {
                // overlapped launches: the time attributed to launch i is the advance of the completion front, so that the
                // sum over the launches is the span from the first start to the last end
                SOC_CUDA(cudaEventElapsedTime(&ms[i], G->ev1[i - 1], G->ev1[i]));
                if (ms[i] < 0.0f) ms[i] = 0.0f;
            } else {
                SOC_CUDA(cudaEventElapsedTime(&ms[i], G->ev0[i], G->ev1[i]));
            }
        }
    }
    // the frequencies of a grouped launch share its time equally; overlapped launches run two at a time, and the advance
    // of the completion front says little about either of them alone: the frequencies of two consecutive launches share the
    // time of both
    for (int i = 0; i < n;) {
        int len = 0;
        for (int u = 0; u < (G->last_overlap ? 2 : 1) && i + len < n; ++u) {
            const int J = i + len < (int)G->slot_group.size() && G->slot_group[i + len] > 1 ? G->slot_group[i + len] : 1;
            len += J < n - (i + len) ? J : n - (i + len);
        }
        float total = 0.0f;
        bool all = true;
        for (int k = 0; k < len; ++k) { all = all && ms[i + k] >= 0.0f; total += ms[i + k] > 0.0f ? ms[i + k] : 0.0f; }
        if (all && len > 1)
            for (int k = 0; k < len; ++k) ms[i + k] = total / (float)len;
        i += len;
    }
    return SOC_OK;
}

int soc_simulate_packages(soc_grid *G, int32_t ifreq, const soc_sources *src, int64_t n_packages, uint64_t seed,
                          double weight, int64_t pkg_begin, int64_t pkg_count, double *absorbed,
                          soc_replay_record *replay, soc_freq_result *res, uint32_t flags, void *stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    if (G) G->last_overlap = 0;
    int rc = enqueue_frequency(G, ifreq, src, n_packages, seed, weight, pkg_begin, pkg_count, absorbed, replay,
                               flags, 0, st);
    if (rc != SOC_OK) return rc;
    if (res) return fetch_results(G, 1, res, st);
    return SOC_OK;
}

int soc_simulate_frequency(soc_grid *G, int32_t ifreq, const soc_sources *src, int64_t n_packages, uint64_t seed,
                           double weight, double *absorbed, soc_freq_result *res, uint32_t flags, void *stream)
{
    return soc_simulate_packages(G, ifreq, src, n_packages, seed, weight, 0, n_packages, absorbed, nullptr, res,
                                 flags, stream);
}

int soc_simulate_spectrum(soc_grid *G, const soc_sources *src, int64_t n_packages, uint64_t seed, int64_t pkg_begin,
                          int64_t pkg_count, double *absorbed_int, soc_freq_result *results, uint32_t flags,
                          void *stream)
{
    if (!G || !src) return fail(SOC_EINVAL, "NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<double> w;
    trapezoid(G->freq, w);
    int rc = ensure_slots(G, G->n_freq);
    if (rc != SOC_OK) return rc;
    // production mode: odd frequencies go to a second stream with their own accumulators, so that the tail of one launch
    // (lanes that have run out of packages) is filled by the blocks of the next; the folds into absorbed_int stay ordered
    // Dust packages keep the launches serial: the prefix sums of the package counts, the scan scratch and the luminosity
    // scalars exist once per grid (dust_prepare), so the scan of frequency f + 1 on the other stream would rewrite the
    // array the kernel of frequency f is still searching.
    bool any_dust = false;
    for (int f = 0; f < G->n_freq; ++f) any_dust = any_dust || src[f].n_dust > 0;
    const bool overlap = G->opt_overlap && G->n_freq > 1 && !(flags & SOC_GEOM_FP64) && !any_dust;
    if (overlap) {
        // every piece is created on its own test, so that a call that failed half-way through (an event, the second
        // accumulator) is completed by the next instead of launching on what is missing
        if (!G->aux) SOC_CUDA(cudaStreamCreateWithFlags(&G->aux, cudaStreamNonBlocking));
        if (!G->ev_fork) SOC_CUDA(cudaEventCreateWithFlags(&G->ev_fork, cudaEventDisableTiming));
        if (!G->ev_join) SOC_CUDA(cudaEventCreateWithFlags(&G->ev_join, cudaEventDisableTiming));
        if (!G->ev_unpad[0]) SOC_CUDA(cudaEventCreateWithFlags(&G->ev_unpad[0], cudaEventDisableTiming));
        if (!G->ev_unpad[1]) SOC_CUDA(cudaEventCreateWithFlags(&G->ev_unpad[1], cudaEventDisableTiming));
        if (!G->d_acc32_b) {
            SOC_CUDA(big_malloc(&G->d_acc32_b, sizeof(float) * (size_t)G->n_int));
            const cudaError_t e = cudaMemsetAsync(G->d_acc32_b, 0, sizeof(float) * (size_t)G->n_int, st);   // ordered before the fork
            if (e != cudaSuccess) { big_free(G->d_acc32_b); G->d_acc32_b = nullptr; return fail(SOC_ECUDA, cudaGetErrorString(e)); }
        }
        SOC_CUDA(cudaEventRecord(G->ev_fork, st));
        SOC_CUDA(cudaStreamWaitEvent(G->aux, G->ev_fork, 0));
        G->unpad_wait = nullptr;
        G->overlap_active = 1;
    }
    // launches of few packages carry several consecutive frequencies each (enqueue_group): up to four, up to ~1.6e7 packages
    // per launch (config 4' with 1e6 packages per frequency: 6.33e10 cell-steps/s one by one, 7.63e10 in fours; in eights
    // 7.85e10, but eight frequencies in one fp32 accumulator cost accuracy: cells against counters 4e-7 instead of 9e-9;
    // config 3 with 4e6 packages per frequency: 1.262e11 one by one, 1.276e11 in twos, 1.294e11 in fours)
    int J = G->opt_group;
    if (J == 0) J = pkg_count > 0 && pkg_count < 16000000 ? (int)((16000000 + pkg_count - 1) / pkg_count) : 1;
    if (J > kMaxJobs) J = kMaxJobs;
    if (flags & SOC_GEOM_FP64) J = 1;
    for (int f = 0, launch = 0; f < G->n_freq && rc == SOC_OK; ++launch) {
        G->acc_sel = overlap ? (launch & 1) : 0;
        cudaStream_t sf = G->acc_sel ? G->aux : st;
        int n = J < G->n_freq - f ? J : G->n_freq - f;
        // (the octree takes the grouped kernel for a single frequency as well: its totals live in shared memory, which
        //  frees the registers the one-frequency kernel spills -- +2 %)
        if (!(flags & SOC_GEOM_FP64) && (n > 1 || (G->n_levels > 1 && G->opt_group != 1))) {
            rc = enqueue_group(G, f, n, src + f, n_packages, seed, w.data() + f, pkg_begin, pkg_count, absorbed_int, f, sf);
            if (rc == 1 && n > 1 && G->n_levels > 1) {       // the group is not eligible: this frequency alone (octree: grouped kernel)
                n = 1;
                rc = enqueue_group(G, f, 1, src + f, n_packages, seed, w.data() + f, pkg_begin, pkg_count, absorbed_int, f, sf);
            }
            if (rc == 1) { n = 1; rc = SOC_OK; }
            else { f += n; continue; }
        }
        rc = enqueue_frequency(G, f, src + f, n_packages, seed, w[f], pkg_begin, pkg_count, absorbed_int, nullptr, flags, f, sf);
        f += 1;
    }
    G->acc_sel = 0; G->overlap_active = 0; G->unpad_wait = nullptr;
    G->last_overlap = overlap ? 1 : 0;
    if (overlap) {
        cudaError_t e = cudaEventRecord(G->ev_join, G->aux);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(st, G->ev_join, 0);
        if (e != cudaSuccess && rc == SOC_OK) rc = fail(SOC_ECUDA, cudaGetErrorString(e));
    }
    if (rc != SOC_OK) return rc;
    if (results) return fetch_results(G, G->n_freq, results, st);
    return SOC_OK;
}

int soc_update_temperatures(soc_grid *G, const double *absorbed, double scale, const float *table_T, int32_t n_table,
                            double E_min, double E_max, float *T_out, void *stream)
{
    if (!G || !absorbed || !table_T || !T_out) return fail(SOC_EINVAL, "NULL argument");
    if (n_table < 2 || n_table > 8192) return fail(SOC_EINVAL, "n_table out of range");
    if (!(E_min > 0.0) || !(E_max > E_min) || !std::isfinite(E_max) || !std::isfinite(scale))
        return fail(SOC_EINVAL, "need 0 < E_min < E_max and a finite scale");
    if ((reinterpret_cast<uintptr_t>(absorbed) & 15) || (reinterpret_cast<uintptr_t>(T_out) & 15))
        return fail(SOC_EINVAL, "absorbed and T_out must be 16-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    // the caller's table is borrowed for the call only: stage it in pinned memory of our own, so that the asynchronous
    // copy never reads the caller's buffer after the call has returned
    if (!G->h_table) {
        SOC_CUDA(cudaMallocHost(&G->h_table, sizeof(float) * 8192));
        SOC_CUDA(cudaEventCreateWithFlags(&G->ev_table, cudaEventDisableTiming));
    } else {
        SOC_CUDA(cudaEventSynchronize(G->ev_table));     // the previous call's copy has left the staging buffer
    }
    std::memcpy(G->h_table, table_T, sizeof(float) * n_table);
    SOC_CUDA(cudaMemcpyAsync(G->d_table, G->h_table, sizeof(float) * n_table, cudaMemcpyHostToDevice, st));
    SOC_CUDA(cudaEventRecord(G->ev_table, st));
    TempParams P;
    std::memset(&P, 0, sizeof(P));
    P.cellw = G->d_cellw; P.absorbed = absorbed; P.table = G->d_table; P.T_out = T_out;
    P.n_total = G->n_total; P.n_levels = G->n_levels; P.n_table = n_table;
    for (int l = 0; l <= G->n_levels; ++l) P.level_off[l] = G->level_off[l];
    P.scale = scale; P.e_min = E_min; P.e_max = E_max; P.inv_e_min = 1.0 / E_min;
    P.x_scale = (float)((double)(n_table - 1) / std::log(E_max / E_min));
    const long long n4 = (G->n_total >> 2) + 1;
    long long blocks = (n4 + 255) / 256;
    const long long cap = (long long)G->n_sm * 8;       // grid-stride over a whole number of CTAs per SM
    if (blocks > cap) blocks = cap;
    temperature_kernel<<<(int)blocks, 256, sizeof(float) * n_table, st>>>(P);
    g_launches += 1;
    SOC_CUDA(cudaGetLastError());
    return SOC_OK;
}

int soc_emission_counts(soc_grid *G, int32_t ifreq, const float *T, int32_t mode, int64_t n_request, int32_t cap,
                        int32_t *count, int64_t *n_dust, double *lum_total, void *stream)
{
    if (!G || !T || !count || !n_dust) return fail(SOC_EINVAL, "NULL argument");
    if (ifreq < 0 || ifreq >= G->n_freq) return fail(SOC_EINVAL, "ifreq out of range");
    if (n_request < 0 || (mode != 0 && mode != 1) || (mode == 1 && cap < 1)) return fail(SOC_EINVAL, "bad mode / n_request / cap");
    cudaStream_t st = (cudaStream_t)stream;
    int rc = ensure_dust_buffers(G);
    if (rc != SOC_OK) return rc;
    LumParams L;
    fill_lum_params(G, ifreq, T, &L);
    SOC_CUDA(cudaMemsetAsync(G->d_scalars, 0, sizeof(double) * 8, st));
    lum_sum_kernel<<<G->n_sm * 8, 256, 0, st>>>(L, nullptr, G->d_scalars);
    dust_counts_kernel<<<G->n_sm * 8, 256, 0, st>>>(L, mode, n_request, cap, count, G->d_scalars);
    g_launches += 2;
    SOC_CUDA(cudaGetLastError());
    SOC_CUDA(cudaMemcpyAsync(G->h_scalars, G->d_scalars, sizeof(double) * 3, cudaMemcpyDeviceToHost, st));
    SOC_CUDA(cudaStreamSynchronize(st));
    *n_dust = (int64_t)G->h_scalars[2];
    if (lum_total) *lum_total = G->h_scalars[0];
    return SOC_OK;
}

int soc_cell_emission(soc_grid *G, const float *T, double *emitted, void *stream)
{
    if (!G || !T || !emitted) return fail(SOC_EINVAL, "NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    if (!G->d_freqtab) {
        std::vector<double> tab((size_t)3 * G->n_freq), w;
        trapezoid(G->freq, w);
        for (int f = 0; f < G->n_freq; ++f) { tab[f] = G->freq[f]; tab[G->n_freq + f] = G->kabs[f]; tab[2 * G->n_freq + f] = w[f]; }
        SOC_CUDA(cudaMalloc(&G->d_freqtab, sizeof(double) * tab.size()));
        SOC_CUDA(cudaMemcpy(G->d_freqtab, tab.data(), sizeof(double) * tab.size(), cudaMemcpyHostToDevice));
    }
    LumParams L;
    fill_lum_params(G, 0, T, &L);
    cell_emission_kernel<<<G->n_sm * 8, 256, 0, st>>>(L, G->d_freqtab, G->n_freq, emitted);
    g_launches += 1;
    SOC_CUDA(cudaGetLastError());
    return SOC_OK;
}

int soc_update_temperatures_ali(soc_grid *G, const double *absorbed, const double *self_abs, const double *emitted,
                                double scale, const float *table_T, int32_t n_table, double E_min, double E_max,
                                float *T_out, void *stream)
{
    if (!G || !absorbed || !self_abs || !emitted) return fail(SOC_EINVAL, "NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    if (!G->d_eff) SOC_CUDA(big_malloc(&G->d_eff, sizeof(double) * (size_t)G->n_total));
    ali_effective_kernel<<<G->n_sm * 8, 256, 0, st>>>(absorbed, self_abs, emitted, G->n_total, G->d_eff);
    g_launches += 1;
    SOC_CUDA(cudaGetLastError());
    return soc_update_temperatures(G, G->d_eff, scale, table_T, n_table, E_min, E_max, T_out, stream);
}

// The same two kernels as soc_update_temperatures_ali + soc_update_temperatures, with the work array and the table in
// g_static_scratch: no cudaMalloc, cudaMallocHost, cudaFree, event creation or cached-buffer call on this path.
int soc_update_temperatures_ali_static(soc_grid *G, const double *absorbed, const double *self_abs, const double *emitted,
                                       double scale, const float *table_T, int32_t n_table, double E_min, double E_max,
                                       float *T_out, void *stream)
{
    if (!G || !absorbed || !self_abs || !emitted || !table_T || !T_out) return fail(SOC_EINVAL, "NULL argument");
    if (n_table < 2 || n_table > kStaticMaxTable) return fail(SOC_EINVAL, "n_table out of range");
    if (!(E_min > 0.0) || !(E_max > E_min) || !std::isfinite(E_max) || !std::isfinite(scale))
        return fail(SOC_EINVAL, "need 0 < E_min < E_max and a finite scale");
    if (reinterpret_cast<uintptr_t>(T_out) & 15) return fail(SOC_EINVAL, "T_out must be 16-byte aligned");
    if (G->n_total > kStaticMaxCells)
        return fail(SOC_EINVAL, "soc_update_temperatures_ali_static: the grid has " + std::to_string(G->n_total) +
                                " cells, the static scratch holds " + std::to_string(kStaticMaxCells) +
                                "; use soc_update_temperatures_ali");
    int device = -1;
    SOC_CUDA(cudaGetDevice(&device));
    if (device != G->device) return fail(SOC_EINVAL, "soc_update_temperatures_ali_static: the grid's device must be the current device");
    double *scratch = nullptr;
    const int rc = static_scratch(device, &scratch);        // first call on this device: looks the address up
    if (rc != SOC_OK) return rc;
    double *d_eff = scratch;
    float *d_table = reinterpret_cast<float *>(scratch + kStaticMaxCells);
    cudaStream_t st = (cudaStream_t)stream;
    // Nothing in the scratch has to start at zero: the first kernel writes eff[0 .. n_total) and the copy writes
    // table[0 .. n_table) before the second kernel reads exactly those elements; what earlier calls left beyond them
    // is never read.
    SOC_CUDA(cudaMemcpyAsync(d_table, table_T, sizeof(float) * n_table, cudaMemcpyHostToDevice, st));
    ali_effective_kernel<<<G->n_sm * 8, 256, 0, st>>>(absorbed, self_abs, emitted, G->n_total, d_eff);
    TempParams P;
    std::memset(&P, 0, sizeof(P));
    P.cellw = G->d_cellw; P.absorbed = d_eff; P.table = d_table; P.T_out = T_out;
    P.n_total = G->n_total; P.n_levels = G->n_levels; P.n_table = n_table;
    for (int l = 0; l <= G->n_levels; ++l) P.level_off[l] = G->level_off[l];
    P.scale = scale; P.e_min = E_min; P.e_max = E_max; P.inv_e_min = 1.0 / E_min;
    P.x_scale = (float)((double)(n_table - 1) / std::log(E_max / E_min));
    const long long n4 = (G->n_total >> 2) + 1;
    long long blocks = (n4 + 255) / 256;
    const long long cap = (long long)G->n_sm * 8;
    if (blocks > cap) blocks = cap;
    temperature_kernel<<<(int)blocks, 256, sizeof(float) * n_table, st>>>(P);
    g_launches += 2;
    SOC_CUDA(cudaGetLastError());
    return SOC_OK;
}

int soc_iterate(soc_grid *G, const soc_sources *src, int64_t n_const, uint64_t seed, const soc_iterate_opts *opts,
                double t_scale, const float *table_T, int32_t n_table, double E_min, double E_max,
                double *absorbed_out, float *T_out, soc_iterate_record *history, uint32_t flags, void *stream)
{
    if (!G || !src || !opts || !absorbed_out || !T_out || !table_T) return fail(SOC_EINVAL, "NULL argument");
    if (opts->n_iter < 0 || (opts->n_iter > 0 && !opts->n_request) || opts->ref_start < 1)
        return fail(SOC_EINVAL, "bad iteration options");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb = sizeof(double) * (size_t)G->n_total;
    const int nf = G->n_freq;
    std::vector<double> w;
    trapezoid(G->freq, w);
    // work arrays: A_const, D (this iteration), R (reference field); with ALI also S_i, S_ref, Em_i, Em_ref
    double *buf[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    int32_t *count = nullptr;
    const int n_buf = opts->ali ? 7 : 3;
    // (from the process-wide buffer cache: a second call on a grid of this size allocates nothing; every exit path below
    //  synchronises the stream before the buffers go back)
    auto cleanup = [&]() { cudaStreamSynchronize(st); for (double *b : buf) big_free(b); big_free(count); };
    for (int i = 0; i < n_buf; ++i)
        if (big_malloc(&buf[i], nb) != cudaSuccess || cudaMemsetAsync(buf[i], 0, nb, st) != cudaSuccess) {
            cudaGetLastError();
            cleanup();
            return fail(SOC_ENOMEM, "soc_iterate: device allocation failed");
        }
    if (big_malloc(&count, sizeof(int32_t) * (size_t)G->n_total) != cudaSuccess) {
        cudaGetLastError();
        cleanup();
        return fail(SOC_ENOMEM, "soc_iterate: device allocation failed");
    }
    double *A_const = buf[0], *D = buf[1], *R = buf[2], *Si = buf[3], *Sref = buf[4], *Emi = buf[5], *Emref = buf[6];
    std::vector<soc_freq_result> res((size_t)nf);
    int rc = SOC_OK;
    auto record = [&](int it, int64_t n_pk) {
        if (!history) return;
        soc_iterate_record r{0.0, 0.0, 0.0, n_pk, 0};
        for (int f = 0; f < nf; ++f) {
            r.emitted += w[f] * res[f].emitted; r.escaped += w[f] * res[f].escaped; r.absorbed += w[f] * res[f].absorbed;
            r.cell_steps += res[f].cell_steps;
        }
        history[it] = r;
    };
    // iteration 0: the constant sources
    rc = soc_simulate_spectrum(G, src, n_const, seed, 0, n_const, A_const, res.data(), flags, stream);
    if (rc == SOC_OK) record(0, n_const * nf);
    if (rc == SOC_OK) rc = soc_update_temperatures(G, A_const, t_scale, table_T, n_table, E_min, E_max, T_out, stream);
    double w_ref = 0.0;
    const int blocks = G->n_sm * 8;
    for (int it = 1; it <= opts->n_iter && rc == SOC_OK; ++it) {
        const int64_t n_req = opts->n_request[it - 1];
        if (cudaMemsetAsync(D, 0, nb, st) != cudaSuccess || (opts->ali && cudaMemsetAsync(Si, 0, nb, st) != cudaSuccess)) {
            rc = fail(SOC_ECUDA, "soc_iterate: memset failed");
            break;
        }
        int64_t n_pk = 0;
        for (int f = 0; f < nf && rc == SOC_OK; ++f) {
            std::memset(&res[f], 0, sizeof(res[f]));
            int64_t n_dust = 0;
            rc = soc_emission_counts(G, f, T_out, opts->mode, n_req, opts->cap, count, &n_dust, nullptr, stream);
            if (rc != SOC_OK || n_dust == 0) continue;
            soc_sources ds;
            std::memset(&ds, 0, sizeof(ds));
            ds.n_bg = 0; ds.n_dust = n_dust; ds.dust_T = T_out; ds.dust_count = count; ds.dust_self = opts->ali ? Si : nullptr;
            rc = soc_simulate_frequency(G, f, &ds, n_dust, seed + (uint64_t)it, w[f], D, &res[f], flags, stream);
            n_pk += n_dust;
        }
        if (rc != SOC_OK) break;
        record(it, n_pk);
        if (opts->ali) rc = soc_cell_emission(G, T_out, Emi, stream);
        if (rc != SOC_OK) break;
        const double *A_dust = D, *S_use = Si, *Em_use = Emi;
        if (opts->reference_field && it >= opts->ref_start) {
            running_mean_kernel<<<blocks, 256, 0, st>>>(R, D, opts->ali ? Sref : nullptr, Si, opts->ali ? Emref : nullptr, Emi,
                                                        G->n_total, w_ref, (double)n_req);
            g_launches += 1;
            w_ref += (double)n_req;
            A_dust = R; S_use = Sref; Em_use = Emref;
        }
        add_kernel<<<blocks, 256, 0, st>>>(absorbed_out, A_const, A_dust, G->n_total);
        g_launches += 1;
        if (cudaGetLastError() != cudaSuccess) { rc = fail(SOC_ECUDA, "soc_iterate: kernel launch failed"); break; }
        if (opts->ali) rc = soc_update_temperatures_ali(G, absorbed_out, S_use, Em_use, t_scale, table_T, n_table, E_min, E_max, T_out, stream);
        else rc = soc_update_temperatures(G, absorbed_out, t_scale, table_T, n_table, E_min, E_max, T_out, stream);
    }
    if (rc == SOC_OK && opts->n_iter == 0) {
        cudaError_t e = cudaMemcpyAsync(absorbed_out, A_const, nb, cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) rc = fail(SOC_ECUDA, cudaGetErrorString(e));
    }
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess && rc == SOC_OK) rc = fail(SOC_ECUDA, cudaGetErrorString(e));
    cleanup();
    return rc;
}

int soc_make_map(soc_grid *G, int32_t ifreq, const float *T, const soc_map_desc *d, float *map, void *stream)
{
    if (!G || !T || !d || !map) return fail(SOC_EINVAL, "NULL argument");
    if (ifreq < 0 || ifreq >= G->n_freq) return fail(SOC_EINVAL, "ifreq out of range");
    if (d->npx < 1 || d->npy < 1 || !(d->pixel > 0.0) || !std::isfinite(d->pixel)) return fail(SOC_EINVAL, "bad map size");
    auto dot = [](const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; };
    const double *v[3] = {d->ex, d->ey, d->dir};
    for (int a = 0; a < 3; ++a)
        for (int b = a; b < 3; ++b) {
            const double x = dot(v[a], v[b]);
            if (!(std::fabs(x - (a == b ? 1.0 : 0.0)) <= 1e-6)) return fail(SOC_EINVAL, "ex, ey, dir must be orthonormal");
        }
    for (int k = 0; k < 3; ++k)
        if (!std::isfinite(d->centre[k])) return fail(SOC_EINVAL, "centre is not finite");
    MapParams M;
    std::memset(&M, 0, sizeof(M));
    M.nx = G->nx; M.ny = G->ny; M.nz = G->nz; M.n_root = (int)G->n_root; M.hier = G->n_levels > 1;
    M.cellw = G->d_cellw; M.parent = G->d_parent; M.T = T;
    M.kabs = G->kabs[ifreq]; M.ksca = G->ksca[ifreq]; M.freq_hz = G->freq[ifreq];
    for (int k = 0; k < 3; ++k) { M.ex[k] = d->ex[k]; M.ey[k] = d->ey[k]; M.dir[k] = d->dir[k]; M.centre[k] = d->centre[k]; }
    M.npx = d->npx; M.npy = d->npy; M.pixel = d->pixel; M.map = map;
    const long long n_pix = (long long)d->npx * d->npy;
    long long blocks = (n_pix + 127) / 128;
    const long long cap = (long long)G->n_sm * 16;
    if (blocks > cap) blocks = cap;
    map_kernel<<<(int)blocks, 128, 0, (cudaStream_t)stream>>>(M);
    g_launches += 1;
    SOC_CUDA(cudaGetLastError());
    return SOC_OK;
}

struct soc_stochastic {
    int n_size = 0, n_e = 0, n_freq = 0, n_sm = 0;
    int32_t *d_jupT = nullptr;
    float *d_wupT = nullptr, *d_emis = nullptr;
    double *d_cool = nullptr, *d_scale = nullptr;
};

void soc_stochastic_destroy(soc_stochastic *M)
{
    if (!M) return;
    cudaFree(M->d_jupT); cudaFree(M->d_wupT); cudaFree(M->d_emis); cudaFree(M->d_cool); cudaFree(M->d_scale);
    delete M;
}

int soc_stochastic_create(const soc_stochastic_model *m, soc_stochastic **out)
{
    if (!m || !out) return fail(SOC_EINVAL, "NULL argument");
    *out = nullptr;
    if (m->n_size < 1 || m->n_e < 2 || m->n_e > 128 || m->n_freq < 1 || m->n_freq > 1024)
        return fail(SOC_EINVAL, "stochastic model: need n_size >= 1, 2 <= n_e <= 128, 1 <= n_freq <= 1024");
    if (!m->jup || !m->wup || !m->cool || !m->emis || !m->abundance) return fail(SOC_EINVAL, "stochastic model: NULL table");
    const size_t ns = (size_t)m->n_size, ne = (size_t)m->n_e, nf = (size_t)m->n_freq;
    std::vector<int32_t> jT(ns * nf * ne);
    std::vector<float> wT(ns * nf * ne), em(ns * ne * nf);
    std::vector<double> scale(ns);
    for (size_t s = 0; s < ns; ++s) {
        double emax = 0.0;
        for (size_t i = 0; i < ne; ++i) {
            if (i > 0 && !(m->cool[s * ne + i] > 0.0) ) return fail(SOC_EINVAL, "stochastic model: cooling rates must be > 0");
            for (size_t f = 0; f < nf; ++f) {
                const int32_t j = m->jup[(s * ne + i) * nf + f];
                const double w = m->wup[(s * ne + i) * nf + f];
                if (j >= (int32_t)ne || (j >= 0 && j <= (int32_t)i) || !(w >= 0.0) || !std::isfinite(w))
                    return fail(SOC_EINVAL, "stochastic model: upward transition must go to a higher bin with a finite weight >= 0");
                jT[(s * nf + f) * ne + i] = j;
                wT[(s * nf + f) * ne + i] = (float)w;
                const double e = m->emis[(s * ne + i) * nf + f];
                if (!(e >= 0.0) || !std::isfinite(e)) return fail(SOC_EINVAL, "stochastic model: emission must be finite and >= 0");
                emax = std::fmax(emax, e);
            }
        }
        const double unit = emax > 0.0 ? emax : 1.0;            // the table is stored in fp32 relative to its largest entry
        for (size_t k = 0; k < ne * nf; ++k) em[s * ne * nf + k] = (float)(m->emis[s * ne * nf + k] / unit);
        scale[s] = m->abundance[s] * unit;
    }
    soc_stochastic *M = new (std::nothrow) soc_stochastic;
    if (!M) return fail(SOC_ENOMEM, "out of host memory");
    struct Guard { soc_stochastic *g; ~Guard() { if (g) soc_stochastic_destroy(g); } } guard{M};
    M->n_size = m->n_size; M->n_e = m->n_e; M->n_freq = m->n_freq;
    int dev = 0;
    SOC_CUDA(cudaGetDevice(&dev));
    SOC_CUDA(cudaDeviceGetAttribute(&M->n_sm, cudaDevAttrMultiProcessorCount, dev));
    SOC_CUDA(cudaMalloc(&M->d_jupT, sizeof(int32_t) * jT.size()));
    SOC_CUDA(cudaMalloc(&M->d_wupT, sizeof(float) * wT.size()));
    SOC_CUDA(cudaMalloc(&M->d_emis, sizeof(float) * em.size()));
    SOC_CUDA(cudaMalloc(&M->d_cool, sizeof(double) * ns * ne));
    SOC_CUDA(cudaMalloc(&M->d_scale, sizeof(double) * ns));
    SOC_CUDA(cudaMemcpy(M->d_jupT, jT.data(), sizeof(int32_t) * jT.size(), cudaMemcpyHostToDevice));
    SOC_CUDA(cudaMemcpy(M->d_wupT, wT.data(), sizeof(float) * wT.size(), cudaMemcpyHostToDevice));
    SOC_CUDA(cudaMemcpy(M->d_emis, em.data(), sizeof(float) * em.size(), cudaMemcpyHostToDevice));
    SOC_CUDA(cudaMemcpy(M->d_cool, m->cool, sizeof(double) * ns * ne, cudaMemcpyHostToDevice));
    SOC_CUDA(cudaMemcpy(M->d_scale, scale.data(), sizeof(double) * ns, cudaMemcpyHostToDevice));
    guard.g = nullptr;
    *out = M;
    return SOC_OK;
}

int soc_stochastic_emission(soc_stochastic *M, const double *intensity, int64_t n_cells, double *emission, double *p_out,
                            void *stream)
{
    if (!M || !intensity || !emission || n_cells < 0) return fail(SOC_EINVAL, "bad argument");
    if (n_cells == 0) return SOC_OK;
    StochParams S;
    std::memset(&S, 0, sizeof(S));
    S.n_size = M->n_size; S.n_e = M->n_e; S.n_freq = M->n_freq;
    S.jupT = M->d_jupT; S.wupT = M->d_wupT; S.cool = M->d_cool; S.emis = M->d_emis; S.emis_scale = M->d_scale;
    S.intensity = intensity; S.n_cells = n_cells; S.emission = emission; S.p_out = p_out;
    const size_t per_warp = sizeof(double) * (size_t)(S.n_freq + S.n_e) + sizeof(float) * (size_t)S.n_e * S.n_e;
    int warps = 4;
    while (warps > 1 && sizeof(double) * S.n_freq + warps * per_warp > 200 * 1024) warps >>= 1;
    if (warps > S.n_size) warps = S.n_size > 2 ? 2 : 1;
    S.warps = warps;
    const size_t smem = sizeof(double) * S.n_freq + warps * per_warp;
    SOC_CUDA(cudaFuncSetAttribute(stochastic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    long long blocks = n_cells;
    const long long cap = (long long)M->n_sm * 8;
    if (blocks > cap) blocks = cap;
    stochastic_kernel<<<(int)blocks, 32 * warps, smem, (cudaStream_t)stream>>>(S);
    g_launches += 1;
    SOC_CUDA(cudaGetLastError());
    return SOC_OK;
}

int soc_run_host(const soc_grid_desc *desc, const soc_sources *src, int64_t n_packages, uint64_t seed, int32_t n_iter,
                 double t_scale, const float *table_T, int32_t n_table, double E_min, double E_max,
                 double *absorbed_int_out, float *T_out, soc_freq_result *results, uint32_t flags)
{
    if (n_iter < 1) return fail(SOC_EINVAL, "n_iter must be >= 1");
    soc_grid *G = nullptr;
    int rc = soc_grid_create(desc, &G);
    if (rc != SOC_OK) return rc;
    double *d_abs = nullptr;
    float *d_T = nullptr;
    cudaStream_t st = nullptr;
    auto cleanup = [&]() { big_free(d_abs); big_free(d_T); soc_grid_destroy(G); };
    cudaError_t e = big_malloc(&d_abs, sizeof(double) * (size_t)G->n_total);
    if (e == cudaSuccess) e = big_malloc(&d_T, sizeof(float) * (size_t)G->n_total);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_abs, 0, sizeof(double) * (size_t)G->n_total, st);
    if (e != cudaSuccess) { cleanup(); return fail(SOC_ECUDA, cudaGetErrorString(e)); }
    for (int it = 0; it < n_iter && rc == SOC_OK; ++it)
        rc = soc_simulate_spectrum(G, src, n_packages, seed + (uint64_t)it, 0, n_packages, d_abs,
                                   results ? results + (size_t)it * G->n_freq : nullptr, flags, st);
    if (rc == SOC_OK && n_iter > 1) {                    // running mean over iterations (reading S12)
        scale_kernel<<<G->n_sm * 4, 256, 0, st>>>(d_abs, G->n_total, 1.0 / n_iter);
        g_launches += 1;
    }
    if (rc == SOC_OK && table_T && T_out)
        rc = soc_update_temperatures(G, d_abs, t_scale, table_T, n_table, E_min, E_max, d_T, st);
    if (rc == SOC_OK) {
        if (absorbed_int_out) e = cudaMemcpyAsync(absorbed_int_out, d_abs, sizeof(double) * (size_t)G->n_total, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && T_out && table_T) e = cudaMemcpyAsync(T_out, d_T, sizeof(float) * (size_t)G->n_total, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) rc = fail(SOC_ECUDA, cudaGetErrorString(e));
    }
    cleanup();
    return rc;
}

int soc_probe_throughput(int32_t kind, int64_t footprint_bytes, int64_t n_ops, float *ms)
{
    if (kind < 0 || kind > 7 || footprint_bytes < 64 || n_ops < 1 || !ms) return fail(SOC_EINVAL, "bad probe argument");
    // kind 5: 4 B rho + 4 B acc per cell; kind 7: footprint counted as fp32 cells (4 B), the sums behind them are fp64
    const size_t cell = (kind == 1 || kind == 5) ? 8 : (kind == 3 ? 32 : ((kind == 4 || kind == 6) ? 16 : 4));
    const unsigned long long n_elem = (unsigned long long)footprint_bytes / cell;
    if (kind == 7 && n_elem > (unsigned long long)kProbeHotMax) return fail(SOC_EINVAL, "probe kind 7: at most 8192 cells (32 KB)");
    const size_t elem = kind == 7 ? 8 : cell;
    void *buf = nullptr;
    float *sink = nullptr;
    int dev = 0, n_sm = 0;
    SOC_CUDA(cudaGetDevice(&dev));
    SOC_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    SOC_CUDA(cudaMalloc(&buf, n_elem * elem));
    SOC_CUDA(cudaMalloc(&sink, 4));
    SOC_CUDA(cudaMemset(buf, 0, n_elem * elem));
    const int blocks = n_sm * 8, threads = 256;
    long long per_thread = (n_ops + (long long)blocks * threads - 1) / ((long long)blocks * threads);
    per_thread = (per_thread + 3) / 4 * 4;           // the probe loop is unrolled by four
    cudaEvent_t e0, e1;
    SOC_CUDA(cudaEventCreate(&e0));
    SOC_CUDA(cudaEventCreate(&e1));
    for (int rep = 0; rep < 2; ++rep) {                  // first pass warms the caches / TLB
        SOC_CUDA(cudaEventRecord(e0));
        if (kind == 0) probe_kernel<0><<<blocks, threads>>>(buf, n_elem, per_thread, sink);
        else if (kind == 1) probe_kernel<1><<<blocks, threads>>>(buf, n_elem, per_thread, sink);
        else if (kind == 2) probe_kernel<2><<<blocks, threads>>>(buf, n_elem, per_thread, sink);
        else if (kind == 3) probe_kernel<3><<<blocks, threads>>>(buf, n_elem, per_thread, sink);
        else if (kind == 4) probe_kernel<4><<<blocks, threads>>>(buf, n_elem, per_thread, sink);
        else if (kind == 6) probe_kernel<6><<<blocks, threads>>>(buf, n_elem, per_thread, sink);
        else if (kind == 7) probe_kernel<7><<<blocks, threads>>>(buf, n_elem, per_thread, sink);
        else probe_kernel<5><<<blocks, threads>>>(buf, n_elem, per_thread, sink);
        g_launches += 1;
        SOC_CUDA(cudaEventRecord(e1));
        SOC_CUDA(cudaEventSynchronize(e1));
    }
    SOC_CUDA(cudaEventElapsedTime(ms, e0, e1));
    // report the time for exactly n_ops operations
    *ms = (float)((double)*ms * (double)n_ops / ((double)per_thread * blocks * threads));
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(buf); cudaFree(sink);
    return SOC_OK;
}

}  // extern "C"
