// hmc_sort.cu -- S1: stable LSD radix sort of fp64 radii carrying the star index.
//
// The paper sorts whole 46-double star records with Quicksort.  Here the
// key is the raw 64-bit pattern of r (order-preserving for positive finite doubles), the payload
// is the 32-bit source index, and the record columns are gathered once at the end by the
// resulting permutation.  Per 8-bit digit one "onesweep" pass: each CTA takes a tile of 4096
// keys in ticket order, ranks them stably inside the tile (warp match + per-warp counters),
// publishes its per-digit counts, obtains the counts of all earlier tiles by decoupled
// look-back, and scatters through shared memory so that global writes are coalesced runs.
// A digit whose histogram has a single occupied bin is skipped.
//
// This general sort is the FALLBACK of S1: hmc_sort_fast.cu sorts ordinary input, and only when it meets a run
// of more than 32 stars agreeing in all the key bits it kept does it raise a device-side flag.  The host cannot
// read that flag without synchronising, so the fallback is always enqueued -- as ONE cooperative launch whose
// CTAs return at once when the flag is clear (round 1 enqueued its 13 kernels separately: 38 us per step of empty
// launches).  Its phases (zero, histograms, bin scan, eight digit passes, identity, column gather) are separated
// by grid-wide barriers.
#include <cooperative_groups.h>
#include "hmc_common.cuh"

namespace hmc {

static constexpr int RADIX_BITS = 8;
static constexpr int RADIX = 1 << RADIX_BITS;
static constexpr int NPASS = 64 / RADIX_BITS;
static constexpr int SORT_THREADS = 256;
static constexpr int SORT_WARPS = SORT_THREADS / 32;
static constexpr int SORT_ITEMS = SORT_TILE / SORT_THREADS;   // 16
static_assert(SORT_THREADS == RADIX, "thread d owns digit d");

// The general sort runs after the fast path of hmc_sort_fast.cu and only if that path met a run
// of near-equal keys it would not resolve (guard[2] != 0).  guard == nullptr: run always.
__device__ __forceinline__ bool guard_open(const uint64_t* __restrict__ guard) { return guard == nullptr || guard[2] != 0; }

// zero-fill of the look-back words, digit histograms and tickets, under the same guard
__device__ __forceinline__ void sort_zero_phase(uint32_t* __restrict__ a, uint64_t na, uint32_t* __restrict__ b, uint64_t nb,
                                                uint32_t* __restrict__ c, uint64_t nc)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x, t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (uint64_t i = t; i < na; i += stride) a[i] = 0;
    for (uint64_t i = t; i < nb; i += stride) b[i] = 0;
    for (uint64_t i = t; i < nc; i += stride) c[i] = 0;
}

static constexpr uint32_t FLAG_AGG = 1u << 30;
static constexpr uint32_t FLAG_INC = 2u << 30;
static constexpr uint32_t FLAG_MASK = 3u << 30;

// ---- digit histograms of all 8 digits in one read -------------------------------------------
// Low digits of a radius are uniformly distributed: plain shared-memory atomics on one of
// HIST_COPIES replicated histograms hardly ever collide.  The two top digits (sign, exponent, top
// mantissa bits) take only a handful of values, so those are first aggregated across the warp.
static constexpr int HIST_THREADS = 256;
static constexpr int HIST_COPIES = 4;
static constexpr int HIST_SKEWED_FROM = 6;      // digits >= this are warp-aggregated

__device__ __forceinline__ void sort_histogram_phase(const uint64_t* __restrict__ keys, uint64_t n,
                                                     uint32_t* __restrict__ hist /*[8][256]*/, unsigned char* smem_raw)
{
    uint32_t (*sh)[NPASS * RADIX] = reinterpret_cast<uint32_t (*)[NPASS * RADIX]>(smem_raw);      // [HIST_COPIES][8 * 256]
    for (int i = threadIdx.x; i < HIST_COPIES * NPASS * RADIX; i += HIST_THREADS) (&sh[0][0])[i] = 0;
    __syncthreads();
    uint32_t* mine = sh[(threadIdx.x >> 5) % HIST_COPIES];
    const uint64_t stride = (uint64_t)gridDim.x * HIST_THREADS;
    const uint64_t iters = (n + stride - 1) / stride;           // same trip count for every thread
    uint64_t i = (uint64_t)blockIdx.x * HIST_THREADS + threadIdx.x;
    for (uint64_t it = 0; it < iters; ++it, i += stride) {
        const bool ok = i < n;
        uint64_t k = ok ? __ldg(keys + i) : 0ull;
        if (ok) {
#pragma unroll
            for (int p = 0; p < HIST_SKEWED_FROM; ++p)
                atomicAdd(&mine[p * RADIX + ((uint32_t)(k >> (p * RADIX_BITS)) & (RADIX - 1))], 1u);
        }
#pragma unroll
        for (int p = HIST_SKEWED_FROM; p < NPASS; ++p) {
            uint32_t d = ok ? ((uint32_t)(k >> (p * RADIX_BITS)) & (RADIX - 1)) : (uint32_t)RADIX;
            unsigned peers = __match_any_sync(0xffffffffu, d);
            if (ok && (peers & lanemask_lt()) == 0) atomicAdd(&mine[p * RADIX + d], __popc(peers));
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < NPASS * RADIX; b += HIST_THREADS) {
        uint32_t c = 0;
#pragma unroll
        for (int q = 0; q < HIST_COPIES; ++q) c += sh[q][b];
        if (c) atomicAdd(&hist[b], c);
    }
}

// exclusive scan of each digit's 256 counts; pass_live[p] = 0 when one bin holds every key
__device__ __forceinline__ void sort_scan_hist_phase(uint32_t* __restrict__ hist, uint64_t n, uint32_t* __restrict__ pass_live,
                                                     int p, unsigned char* smem_raw)
{
    uint32_t* sh = reinterpret_cast<uint32_t*>(smem_raw);                                         // [256]
    const int d = threadIdx.x;
    __syncthreads();
    uint32_t c = hist[p * RADIX + d];
    sh[d] = c;
    __syncthreads();
    // Hillis-Steele inclusive scan over 256 counts
    for (int off = 1; off < RADIX; off <<= 1) {
        uint32_t v = (d >= off) ? sh[d - off] : 0;
        __syncthreads();
        sh[d] += v;
        __syncthreads();
    }
    hist[p * RADIX + d] = sh[d] - c;
    int single = __syncthreads_or(c == (uint32_t)n);
    if (d == 0) pass_live[p] = single ? 0u : 1u;
}

// ---- one onesweep pass ----------------------------------------------------------------------
struct SortSmem {
    uint64_t keys[SORT_TILE];
    uint32_t vals[SORT_TILE];
    uint32_t warp_counts[SORT_WARPS][RADIX];
    uint32_t digit_base[RADIX];      // exclusive offset of digit d inside the tile
    uint32_t global_base[RADIX];     // where digit d of this tile starts in the output, minus digit_base
    uint32_t tile;
};

// Which passes are live (digit not constant) is known only on the device, and the host must not
// synchronise, so every pass picks its own buffers: the i-th of L live passes reads the source
// keys (i == 0) or the output of live pass i-1, and writes buffer 1 ^ ((L-1-i) & 1); buffer 1 is
// the caller's (r_sorted, perm), so the last live pass always lands there.  A pass whose digit is
// constant returns at once and moves no data.
struct SortBuffers {
    const uint64_t* keys_src;   // the caller's r_in
    uint64_t* keys[2];
    uint32_t* vals[2];
};

__device__ __forceinline__ void sort_onesweep_phase(const SortBuffers& buf, uint32_t n, int shift,
                                                    const uint32_t* __restrict__ bin_offset /*[256] exclusive*/,
                                                    uint32_t* __restrict__ lookback, uint32_t* __restrict__ ticket,
                                                    const uint32_t* __restrict__ pass_live, int pass, unsigned char* smem_raw)
{
    if (!pass_live[pass]) return;
    int live_before = 0, live_total = 0;
#pragma unroll
    for (int p = 0; p < NPASS; ++p) {
        int l = pass_live[p] ? 1 : 0;
        live_total += l;
        if (p < pass) live_before += l;
    }
    const bool FIRST_PASS = live_before == 0;
    const int ob = 1 ^ ((live_total - 1 - live_before) & 1);
    const uint64_t* __restrict__ keys_in = FIRST_PASS ? buf.keys_src : buf.keys[ob ^ 1];
    const uint32_t* __restrict__ vals_in = buf.vals[ob ^ 1];
    uint64_t* __restrict__ keys_out = buf.keys[ob];
    uint32_t* __restrict__ vals_out = buf.vals[ob];
    SortSmem& s = *reinterpret_cast<SortSmem*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // persistent CTAs: tiles are taken in ticket order until none is left
    const uint32_t tiles = (n + SORT_TILE - 1) / SORT_TILE;
    for (;;) {
    __syncthreads();                                            // previous tile's shared memory is no longer read
    if (tid == 0) s.tile = atomicAdd(ticket, 1u);
    for (int i = tid; i < SORT_WARPS * RADIX; i += SORT_THREADS) (&s.warp_counts[0][0])[i] = 0;
    __syncthreads();
    const uint32_t tile = s.tile;
    if (tile >= tiles) break;
    const uint32_t tile_base = tile * SORT_TILE;
    const uint32_t valid = min((uint32_t)SORT_TILE, n - tile_base);

    // load, warp-striped: item i of lane l sits at tile position warp*512 + i*32 + l
    uint64_t key[SORT_ITEMS];
    uint32_t val[SORT_ITEMS];
    uint32_t rank[SORT_ITEMS];
    const uint32_t wbase = warp * (32 * SORT_ITEMS) + lane;
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; ++i) {
        uint32_t pos = wbase + i * 32;
        bool ok = pos < valid;
        key[i] = ok ? keys_in[tile_base + pos] : ~0ull;     // padding sorts last inside the tile
        val[i] = FIRST_PASS ? (tile_base + pos) : (ok ? vals_in[tile_base + pos] : 0u);
    }

    // stable rank inside the warp, digit by digit (items in order, lanes in order)
    uint32_t* wc = s.warp_counts[warp];
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; ++i) {
        uint32_t d = (uint32_t)(key[i] >> shift) & (RADIX - 1);
        unsigned peers = __match_any_sync(0xffffffffu, d);
        int leader = __ffs(peers) - 1;
        uint32_t before = 0;
        if (lane == leader) { before = wc[d]; wc[d] = before + __popc(peers); }
        before = __shfl_sync(0xffffffffu, before, leader);
        rank[i] = before + __popc(peers & lanemask_lt());
        __syncwarp();
    }
    __syncthreads();

    // thread d owns digit d: offsets of each warp's share, the tile count, look-back
    {
        const int d = tid;
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) { uint32_t c = s.warp_counts[w][d]; s.warp_counts[w][d] = run; run += c; }
        uint32_t count = run;
        if (tile_base + SORT_TILE > n && d == RADIX - 1) count -= (SORT_TILE - valid);   // padding is not data
        // publish the aggregate, then sum the aggregates of earlier tiles
        uint32_t* my = lookback + (size_t)tile * RADIX + d;
        st_volatile_u32(my, FLAG_AGG | count);
        uint32_t excl = 0;
        for (int64_t t = (int64_t)tile - 1; t >= 0; --t) {
            const uint32_t* q = lookback + (size_t)t * RADIX + d;
            uint32_t v;
            do { v = ld_volatile_u32(q); } while ((v & FLAG_MASK) == 0);
            excl += v & ~FLAG_MASK;
            if ((v & FLAG_MASK) == FLAG_INC) break;
        }
        st_volatile_u32(my, FLAG_INC | (excl + count));
        // block-wide exclusive scan of the (padded) tile counts -> position of digit d in the tile
        s.digit_base[d] = run;
        __syncthreads();
        for (int off = 1; off < RADIX; off <<= 1) {
            uint32_t v = (d >= off) ? s.digit_base[d - off] : 0;
            __syncthreads();
            s.digit_base[d] += v;
            __syncthreads();
        }
        uint32_t base = s.digit_base[d] - run;    // exclusive
        __syncthreads();
        s.digit_base[d] = base;
        s.global_base[d] = bin_offset[d] + excl - base;
    }
    __syncthreads();

    // scatter into shared memory at the tile-sorted position
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; ++i) {
        uint32_t d = (uint32_t)(key[i] >> shift) & (RADIX - 1);
        uint32_t pos = s.digit_base[d] + s.warp_counts[warp][d] + rank[i];
        s.keys[pos] = key[i];
        s.vals[pos] = val[i];
    }
    __syncthreads();
    // coalesced runs to global memory
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; ++i) {
        uint32_t pos = tid + i * SORT_THREADS;
        if (pos < valid) {
            uint64_t k = s.keys[pos];
            uint32_t d = (uint32_t)(k >> shift) & (RADIX - 1);
            uint32_t g = s.global_base[d] + pos;
            keys_out[g] = k;
            vals_out[g] = s.vals[pos];
        }
    }
    }   // tile loop
}

// ---- copy-through for the degenerate case "every pass skipped" and final gather ---------------
__device__ __forceinline__ void sort_iota_copy_phase(const uint64_t* __restrict__ keys_in, uint64_t* __restrict__ keys_out,
                                                     uint32_t* __restrict__ perm, uint64_t n, const uint32_t* __restrict__ pass_live)
{
    // does something only when no pass was live (all keys equal): identity permutation
    uint32_t any = 0;
    for (int p = 0; p < NPASS; ++p) any |= pass_live[p];
    if (any) return;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        keys_out[i] = keys_in[i];
        perm[i] = (uint32_t)i;
    }
}

struct GatherCols {
    const double* in[HMC_MAX_COLS];
    double* out[HMC_MAX_COLS];
    const uint32_t* id_in;
    uint32_t* id_out;
    int ncols;
};

__device__ __forceinline__ void sort_gather_phase(const GatherCols& g, const uint32_t* __restrict__ perm, uint64_t n)
{
    if (g.ncols == 0 && !g.id_in) return;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += stride) {
        uint32_t src = perm[k];
        double v[HMC_MAX_COLS];
#pragma unroll
        for (int c = 0; c < HMC_MAX_COLS; ++c)
            if (c < g.ncols) v[c] = __ldg(g.in[c] + src);
        uint32_t idv = g.id_in ? __ldg(g.id_in + src) : 0u;
#pragma unroll
        for (int c = 0; c < HMC_MAX_COLS; ++c)
            if (c < g.ncols) g.out[c][k] = v[c];
        if (g.id_out) g.id_out[k] = idv;
    }
}

hmc_status sort_fast(uint64_t n, const double* r_in, double* r_sorted, uint32_t* perm, int ncols,
                     const double* const* cols_in, double* const* cols_out, const uint32_t* id_in, uint32_t* id_out,
                     const Workspace& ws, cudaStream_t st);

// ---- the whole general sort as one cooperative launch ------------------------------------------------
struct GeneralSortArgs {
    SortBuffers buf;
    GatherCols cols;
    uint32_t *lookback, *digit_hist, *tickets;   // tickets: [0..7] tile tickets, [8..15] pass_live
    uint32_t* perm;
    const uint64_t* guard;                       // sortctl of the fast path, or nullptr: run always
    uint64_t n;
    uint32_t tiles;
};

static constexpr size_t GENERAL_SMEM = sizeof(SortSmem) > HIST_COPIES * NPASS * RADIX * 4 ? sizeof(SortSmem) : HIST_COPIES * NPASS * RADIX * 4;

__global__ void __launch_bounds__(SORT_THREADS, 2) sort_general_kernel(GeneralSortArgs a)
{
    if (!guard_open(a.guard)) return;                            // the same answer in every CTA: nobody waits at a barrier
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    uint32_t* pass_live = a.tickets + 8;
    sort_zero_phase(a.lookback, (uint64_t)NPASS * a.tiles * RADIX, a.digit_hist, NPASS * RADIX, a.tickets, 16);
    grid.sync();
    sort_histogram_phase(a.buf.keys_src, a.n, a.digit_hist, smem_raw);
    grid.sync();
    for (int p = blockIdx.x; p < NPASS; p += gridDim.x) sort_scan_hist_phase(a.digit_hist, a.n, pass_live, p, smem_raw);
    grid.sync();
    for (int p = 0; p < NPASS; ++p) {
        sort_onesweep_phase(a.buf, (uint32_t)a.n, p * RADIX_BITS, a.digit_hist + p * RADIX, a.lookback + (size_t)p * a.tiles * RADIX,
                            a.tickets + p, pass_live, p, smem_raw);
        grid.sync();
    }
    sort_iota_copy_phase(a.buf.keys_src, a.buf.keys[1], a.perm, a.n, pass_live);
    grid.sync();
    sort_gather_phase(a.cols, a.perm, a.n);
}

// CTAs that can be resident at once on the current device (a cooperative launch must not exceed it)
static hmc_status general_grid_limit(int* out)
{
    static std::atomic<int> cached[64];
    int dev = 0;
    HMC_CUDA_TRY(cudaGetDevice(&dev));
    const bool slot = dev >= 0 && dev < 64;
    int v = slot ? cached[dev].load(std::memory_order_relaxed) : 0;
    if (v <= 0) {
        int per_sm = 0;
        HMC_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, sort_general_kernel, SORT_THREADS, GENERAL_SMEM));
        if (per_sm < 1) return HMC_ERR_CUDA;
        v = (per_sm > 2 ? 2 : per_sm) * sm_count();
        if (slot) cached[dev].store(v, std::memory_order_relaxed);
    }
    *out = v;
    return HMC_OK;
}

// the general eight-pass sort; with a guard it is enqueued but does nothing unless the guard is set
static hmc_status sort_general(uint64_t n, const double* r_in, double* r_sorted, uint32_t* perm, int ncols,
                               const double* const* cols_in, double* const* cols_out, const uint32_t* id_in,
                               uint32_t* id_out, const Workspace& ws, const uint64_t* guard, cudaStream_t st)
{
    static std::atomic<uint64_t> opted{ 0 };
    hmc_status so = smem_opt_in(opted, sort_general_kernel, GENERAL_SMEM);
    if (so != HMC_OK) return so;
    int limit = 0;
    so = general_grid_limit(&limit);
    if (so != HMC_OK) return so;
    GeneralSortArgs a{};
    a.tiles = (uint32_t)((n + SORT_TILE - 1) / SORT_TILE);
    a.n = n;
    a.buf.keys_src = reinterpret_cast<const uint64_t*>(r_in);
    a.buf.keys[0] = ws.keys_alt; a.buf.keys[1] = reinterpret_cast<uint64_t*>(r_sorted);
    a.buf.vals[0] = ws.vals_alt; a.buf.vals[1] = perm;
    a.cols.ncols = ncols;
    for (int c = 0; c < ncols; ++c) { a.cols.in[c] = cols_in[c]; a.cols.out[c] = cols_out[c]; }
    a.cols.id_in = id_in; a.cols.id_out = id_out;
    a.lookback = ws.lookback; a.digit_hist = ws.digit_hist; a.tickets = ws.tickets;
    a.perm = perm;
    a.guard = guard;
    const unsigned blocks = (unsigned)umin64(a.tiles > 8 ? a.tiles : 8, (uint64_t)limit);
    void* args[] = { &a };
    HMC_CUDA_TRY(cudaLaunchCooperativeKernel(reinterpret_cast<void*>(sort_general_kernel), dim3(blocks), dim3(SORT_THREADS), args,
                                             GENERAL_SMEM, st));
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

__global__ void __launch_bounds__(256) sort_gather_kernel(GatherCols g, const uint32_t* __restrict__ perm, uint64_t n)
{
    sort_gather_phase(g, perm, n);
}

hmc_status gather_by_perm(uint64_t n, const uint32_t* perm, int ncols, const double* const* cols_in, double* const* cols_out,
                          const uint32_t* id_in, uint32_t* id_out, cudaStream_t st)
{
    if (n == 0 || (ncols == 0 && !id_in)) return HMC_OK;
    GatherCols g{};
    g.ncols = ncols;
    for (int c = 0; c < ncols; ++c) { g.in[c] = cols_in[c]; g.out[c] = cols_out[c]; }
    g.id_in = id_in; g.id_out = id_out;
    sort_gather_kernel<<<(int)umin64((n + 255) / 256, (uint64_t)sm_count() * 8), 256, 0, st>>>(g, perm, n);
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

hmc_status sort_by_radius(uint64_t n, const double* r_in, double* r_sorted, uint32_t* perm, int ncols,
                          const double* const* cols_in, double* const* cols_out, const uint32_t* id_in,
                          uint32_t* id_out, const Workspace& ws, cudaStream_t st)
{
    if (n < 2) return sort_general(n, r_in, r_sorted, perm, ncols, cols_in, cols_out, id_in, id_out, ws, nullptr, st);
    hmc_status s = sort_fast(n, r_in, r_sorted, perm, ncols, cols_in, cols_out, id_in, id_out, ws, st);
    if (s != HMC_OK) return s;
    return sort_general(n, r_in, r_sorted, perm, ncols, cols_in, cols_out, id_in, id_out, ws, ws.sortctl, st);
}

}  // namespace hmc
