// hmc_common.cuh -- shared by the kernels of libhmc (sm_100a only).
// Compiled with -fmad=false: every fp64 +,-,*,/,sqrt below is one IEEE-754 operation in the
// order written (R2).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <atomic>
#include "hmc.h"

#define HMC_SM_COUNT_FALLBACK 148

namespace hmc {

// One entry of the node table the orbit kernels search: node j (paper numbering, 0..N+1) holds
// r_j, Phi_j, B_j = G M_j and u_j = 1/r_j -- everything Eq. 6 and the in-shell quadratic need, in
// one 32-byte sector.  Sentinels: node 0 = (0, Phi_1, 0, 0), node N+1 = (+inf, 0, G M_N, 0).
struct __align__(32) Node { double r, phi, B, u; };

// ---- host-side checks ---------------------------------------------------------------------
static inline bool misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) != 0; }

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

static inline uint64_t umin64(uint64_t a, uint64_t b) { return a < b ? a : b; }

static inline hmc_status cuda_ok(cudaError_t e) { return e == cudaSuccess ? HMC_OK : HMC_ERR_CUDA; }

#define HMC_CUDA_TRY(expr)                                   \
    do {                                                     \
        cudaError_t _e = (expr);                             \
        if (_e != cudaSuccess) return HMC_ERR_CUDA;          \
    } while (0)

// after every kernel launch: counts it (hmc_launch_count) and turns a launch failure into HMC_ERR_CUDA
#define HMC_LAUNCH_CHECK()                                   \
    do {                                                     \
        ::hmc::g_launches.fetch_add(1, std::memory_order_relaxed); \
        if (cudaPeekAtLastError() != cudaSuccess) return HMC_ERR_CUDA; \
    } while (0)

extern std::atomic<uint64_t> g_launches;   // kernels launched by this process through the library

int sm_count();   // multiprocessor count of the CURRENT device (cached per device)

// Function attributes (the opt-in to more than 48 KB of dynamic shared memory) are per DEVICE: a kernel's
// attribute is set the first time the kernel is launched on each device.  `mask` has one bit per device
// ordinal < 64 (beyond that the attribute is simply set every time); setting it twice is harmless, so no lock.
template <class Kernel>
static inline hmc_status smem_opt_in(std::atomic<uint64_t>& mask, Kernel kernel, size_t bytes)
{
    int dev = 0;
    HMC_CUDA_TRY(cudaGetDevice(&dev));
    if (dev >= 0 && dev < 64 && ((mask.load(std::memory_order_acquire) >> dev) & 1ull)) return HMC_OK;
    HMC_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    if (dev >= 0 && dev < 64) mask.fetch_or(1ull << dev, std::memory_order_release);
    return HMC_OK;
}

// ---- workspace layout (one carve-up used by every call) -------------------------------------
// All offsets are multiples of 256 bytes.
struct Workspace {
    // sort
    uint64_t* keys_alt;      // [n]
    uint32_t* vals_alt;      // [n]
    uint32_t* digit_hist;    // [8][256] global digit counts -> exclusive bin offsets
    uint32_t* lookback;      // [8][sort_tiles][256] tile status words
    uint32_t* tickets;       // [32]: sort tile tickets 0..7, sort pass_live 8..15, scan tickets 16..17
    // sort, fast path (packed words, hmc_sort_fast.cu)
    uint64_t* pk_alt;        // [n] second packed-word buffer (the first is keys_alt)
    unsigned char* rec;      // [n] 64-byte star records (r, columns, id)
    uint64_t* sortctl;       // [8]: key minimum, key maximum, long-run flag
    uint32_t* pk_hist;       // [5][256]
    uint32_t* pk_tickets;    // [16]: tile tickets 0..4, pass_live 8..12
    // potential
    double*   scan_status;   // [2][scan_tiles][8] (flag, agg_hi, agg_lo, inc_hi, inc_lo, pad)
    // orbit
    Node*     nodes;         // [n + 2] node table with sentinels (hmc_orbit.cu)
    uint32_t* dir;           // radius directory, dir_entries(n) entries (hmc_orbit.cu)
    double2*  mid;           // [(n >> MID_SHIFT) + 2] (r, Phi) of every 1024-th node (hmc_orbit.cu, large n only)
    double*   orbitF;        // [n] S3's rejection bound F per star, read by S4 with reuse_tables (hmc_orbit.cu)
    double2*  coarse;        // [COARSE_CAP] (r, Phi) of every 2^shift-th node, contiguous (hmc_orbit.cu)
    size_t    total;
};

// ---- orbit tables: sizes shared by carve() and hmc_orbit.cu ---------------------------------
static constexpr int MID_SHIFT = 10;                 // S3's second search table: every 1024-th node, used when the coarse spacing is wider
static constexpr uint32_t COARSE_CAP = 10240;        // (r, Phi) pairs of the shared-memory coarse table: 160 KB

// coarse nodes are the multiples of 2^shift; smallest shift with (n >> shift) + 2 <= COARSE_CAP
static inline int coarse_shift(uint64_t n)
{
    int t = 0;
    while ((n >> t) + 2 > COARSE_CAP) ++t;
    return t;
}

// the directory holds, for each of the (n >> shift) + 1 coarse intervals, 2^shift 32-bit entries
static inline uint64_t dir_entries(uint64_t n)
{
    const int t = coarse_shift(n);
    return ((n >> t) + 1) * (1ull << t);
}

static constexpr int SORT_TILE = 4096;     // keys per sort tile
static constexpr int SCAN_TILE = 2048;     // elements per scan tile

static inline Workspace carve(void* base, uint64_t n)
{
    Workspace w;
    char* p = static_cast<char*>(base);
    size_t off = 0;
    const uint64_t sort_tiles = (n + SORT_TILE - 1) / SORT_TILE;
    const uint64_t scan_tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    auto take = [&](size_t bytes) { char* q = p ? p + off : nullptr; off += align_up(bytes, 256); return q; };
    w.keys_alt    = reinterpret_cast<uint64_t*>(take(n * 8));
    w.vals_alt    = reinterpret_cast<uint32_t*>(take(n * 4));
    w.digit_hist  = reinterpret_cast<uint32_t*>(take(8 * 256 * 4));
    w.lookback    = reinterpret_cast<uint32_t*>(take(16 * sort_tiles * 256 * 4));   // enough for 5 passes over tiles of 1024
    w.tickets     = reinterpret_cast<uint32_t*>(take(32 * 4));
    w.pk_alt      = reinterpret_cast<uint64_t*>(take(n * 8));
    w.rec         = reinterpret_cast<unsigned char*>(take(n * 64));
    w.sortctl     = reinterpret_cast<uint64_t*>(take(8 * 8));
    w.pk_hist     = reinterpret_cast<uint32_t*>(take(5 * 256 * 4));
    w.pk_tickets  = reinterpret_cast<uint32_t*>(take(16 * 4));
    w.scan_status = reinterpret_cast<double*>(take(2 * scan_tiles * 8 * 8));
    w.nodes       = reinterpret_cast<Node*>(take((n + 2) * sizeof(Node)));
    w.dir         = reinterpret_cast<uint32_t*>(take(dir_entries(n) * 4));
    w.coarse      = reinterpret_cast<double2*>(take(COARSE_CAP * sizeof(double2)));
    w.orbitF      = reinterpret_cast<double*>(take(n * 8));
    w.mid         = reinterpret_cast<double2*>(take(((n >> MID_SHIFT) + 2) * sizeof(double2)));
    w.total = off;
    return w;
}

#ifdef __CUDACC__
// ---- double-double arithmetic (error-free transformations; needs -fmad=false) ---------------
struct dd { double hi, lo; };

__device__ __forceinline__ dd two_sum(double a, double b)
{
    double s = a + b;
    double bb = s - a;
    double e = (a - (s - bb)) + (b - bb);
    return dd{ s, e };
}

__device__ __forceinline__ dd quick_two_sum(double a, double b)   // requires |a| >= |b|
{
    double s = a + b;
    double e = b - (s - a);
    return dd{ s, e };
}

// accurate double-double addition (both components through two_sum), result normalised:
// |lo| <= ulp(hi)/2, so hi is the double-double value rounded to nearest binary64.
__device__ __forceinline__ dd dd_add(dd a, dd b)
{
    dd s = two_sum(a.hi, b.hi);
    dd t = two_sum(a.lo, b.lo);
    s.lo += t.hi;
    s = quick_two_sum(s.hi, s.lo);
    s.lo += t.lo;
    return quick_two_sum(s.hi, s.lo);
}

__device__ __forceinline__ dd dd_add_d(dd a, double b)
{
    dd s = two_sum(a.hi, b);
    s.lo += a.lo;
    return quick_two_sum(s.hi, s.lo);
}

__device__ __forceinline__ dd dd_shfl_up(dd v, int delta)
{
    return dd{ __shfl_up_sync(0xffffffffu, v.hi, delta), __shfl_up_sync(0xffffffffu, v.lo, delta) };
}

// ---- memory helpers -------------------------------------------------------------------------
__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t* p)
{
    uint32_t v;
    asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ double ld_volatile_f64(const double* p)
{
    double v;
    asm volatile("ld.volatile.global.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_volatile_f64(double* p, double v)
{
    asm volatile("st.volatile.global.f64 [%0], %1;" ::"l"(p), "d"(v));
}
__device__ __forceinline__ void st_volatile_u32(uint32_t* p, uint32_t v)
{
    asm volatile("st.volatile.global.u32 [%0], %1;" ::"l"(p), "r"(v));
}

__device__ __forceinline__ unsigned lanemask_lt()
{
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}
// ---- Philox4x32-10 (Salmon et al. 2011) ---------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t w[4])
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
}

// ((hi * 2^32 + lo) >> 11) * 2^-53, a double in [0, 1) (R9).  The 53-bit integer is split into its top 21 and
// low 32 bits, converted separately (both exact) and added (exact: 53 bits): the same value as converting the 64-bit
// integer, without the slow 64-bit integer-to-double conversion.
__device__ __forceinline__ double u53_to_unit(uint32_t hi, uint32_t lo)
{
    const double two_m21 = 1.0 / 2097152.0, two_m53 = 1.0 / 9007199254740992.0;
    return __uint2double_rn(hi >> 11) * two_m21 + __uint2double_rn((hi << 21) | (lo >> 11)) * two_m53;
}
#endif  // __CUDACC__

// stage entry points implemented in the .cu files (same signatures as hmc.h, Workspace carved)
hmc_status sort_by_radius(uint64_t n, const double* r_in, double* r_sorted, uint32_t* perm, int ncols,
                          const double* const* cols_in, double* const* cols_out, const uint32_t* id_in,
                          uint32_t* id_out, const Workspace& ws, cudaStream_t st);
// ext_tot == nullptr: the whole cluster.  Else (sharded step): r, m are shard `rank` of `nranks` consecutive shards of
// the sorted cluster and ext_tot[nranks][4] (device) holds every shard's totals as potential_totals() writes them.
// cols_out[c][k] = cols_in[c][perm[k]] (and the ids likewise): the record columns when they arrive after the sort
hmc_status gather_by_perm(uint64_t n, const uint32_t* perm, int ncols, const double* const* cols_in, double* const* cols_out,
                          const uint32_t* id_in, uint32_t* id_out, cudaStream_t st);
// npeers > 0: the shard's r, phi and m_cum are also stored to peer_*[g] (each already offset to the shard's place)
hmc_status potential(uint64_t n, double G, const double* r, const double* m, double* phi, double* m_cum,
                     const double* ext_tot, uint32_t nranks, uint32_t rank, const Workspace& ws, cudaStream_t st,
                     int npeers = 0, double* const* peer_r = nullptr, double* const* peer_phi = nullptr,
                     double* const* peer_m_cum = nullptr);
hmc_status potential_totals(uint64_t n, const double* r, const double* m, double* totals4, const Workspace& ws, cudaStream_t st);
hmc_status partition_points(uint64_t n, const double* r_sorted, uint32_t nsplit, const double* splitters, uint64_t* counts,
                            cudaStream_t st);
// orbit stages: the table arrays (r, phi, m_cum) are [n]; the stars treated are positions first .. first+count-1 of
// the table and every per-star array is [count] (the single-GPU calls pass first = 0, count = n)
hmc_status turning_points(uint64_t n, uint64_t first, uint64_t count, double G, const double* r, const double* v_r, const double* v_t,
                          const double* phi, const double* m_cum, double* E, double* J, double* r_min,
                          double* r_max, uint32_t* k_min, uint32_t* k_max, uint8_t* status, uint64_t* counters,
                          const Workspace& ws, cudaStream_t st, bool reuse_tables = false);
hmc_status orbit_build_tables(uint64_t n, double G, const double* r, const double* phi, const double* m_cum, const Workspace& ws,
                              cudaStream_t st);
hmc_status sample_new_radius(uint64_t n, uint64_t first, uint64_t count, double G, uint64_t seed, uint32_t step, const double* r,
                             const double* phi, const double* m_cum, const double* v_r, const double* v_t,
                             const double* E, const double* J, const double* r_min, const double* r_max,
                             const uint32_t* k_min, const uint32_t* k_max, const uint32_t* id,
                             const uint8_t* status_in, double* r_new, double* v_r_new, double* v_t_new,
                             uint16_t* n_try, uint8_t* status_out, uint64_t* counters, bool reuse_tables,
                             const Workspace& ws, cudaStream_t st, const uint32_t* step_dev = nullptr);
hmc_status add_u32(uint32_t* p, uint32_t inc, cudaStream_t st);

hmc_status orbit_step(uint64_t n, uint64_t first, uint64_t count, double G, uint64_t seed, uint32_t step, const double* r, const double* v_r,
                      const double* v_t, const double* phi, const double* m_cum, const uint32_t* id, double* E,
                      double* J, double* r_min, double* r_max, uint32_t* k_min, uint32_t* k_max, uint8_t* status,
                      double* r_new, double* v_r_new, double* v_t_new, uint16_t* n_try, uint8_t* status_out,
                      uint64_t* counters, const Workspace& ws, cudaStream_t st);

hmc_status energy_correction(uint64_t n, double G, const double* r, const double* phi, const double* m_cum,
                             const double* E_old, const double* r_old, const double* p_old, const double* v_r,
                             const double* v_t, double* v_r_out, double* v_t_out, uint8_t* status_out,
                             uint64_t* counters, const Workspace& ws, cudaStream_t st);
hmc_status relaxation_timestep(uint64_t n, double G, double ln_gamma_n, double theta_max, const double* r, const double* v_r,
                               const double* v_t, const double* m, double* t_rel_bin, double* t_rel_min, const Workspace& ws,
                               cudaStream_t st);
hmc_status two_body_relaxation(uint64_t n, double G, double ln_gamma_n, double dt, const double* dt_dev, uint64_t seed, uint32_t step, const double* r,
                               const double* v_r, const double* v_t, const double* m, const uint32_t* id, double* v_r_out,
                               double* v_t_out, cudaStream_t st);
hmc_status diagnostics(uint64_t n, double G, const double* r, const double* v_r, const double* v_t, const double* m,
                       const double* phi, const double* m_cum, int nfrac, const double* fractions, double* out,
                       const Workspace& ws, cudaStream_t st);

}  // namespace hmc
