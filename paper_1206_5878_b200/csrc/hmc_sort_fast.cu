// hmc_sort_fast.cu -- S1, the path taken on ordinary input.
//
// The order wanted is the unique one by the pair (r_i, i).  Sorting full 64-bit keys plus an index
// costs eight digit passes over 12 bytes per star.  Here each star is one 64-bit word
//
//      w_i = ((bits(r_i) - kmin) >> s) << IB  |  i          IB = index bits (24, more if n > 2^24)
//
// kmin = smallest key, s = how many low key bits do not fit beside the index (0 when the keys span
// fewer than 64 - IB bits; a narrower span is shifted up instead, so that it fills the kept bits).  The word keeps
// up to 40 key bits, but the stable LSD radix sort runs only over the leading SB = 16, 24 or 32 of them (about
// log2 N: three 8-bit passes at N = 1e7 instead of the four that sorting every kept bit took): that orders the
// stars up to RUNS that agree in those leading bits -- about ten stars long where a Plummer cluster is densest --
// and the rest of the order is already in the word: inside a run, whole words compare as (key bits, index).  The
// final kernel, which also carries the record columns to their sorted places, detects each run from the neighbouring
// words (coalesced, no extra memory traffic) and ranks every member inside it; only members that agree in ALL kept
// key bits while low bits were dropped (s > 0: a handful per million) need their full keys read.  A run longer
// than RUN_MAX sets a flag instead, and the general eight-pass sort of hmc_sort.cu, which is launched
// after this path and returns at once when the flag is clear, redoes the call.
//
// Record columns: one random 8-byte read per column per star costs a whole DRAM line each.
// The columns are therefore first copied, coalesced, into one 64-byte record per star
// (r, columns, id) -- by the histogram kernel, which reads the radii anyway and is bound by
// shared-memory atomics, not by memory -- and the final kernel fetches one record per star.
#include "hmc_common.cuh"

namespace hmc {

static constexpr int PK_RADIX = 256;
static constexpr int PK_MAXPASS = 5;
static constexpr int PK_KEYBITS_MAX = 40;
static constexpr int PK_THREADS = 512;
static constexpr int PK_WARPS = PK_THREADS / 32;
static constexpr int PK_ITEMS = 8;                             // words per thread and tile (6: 3 % slower, 12 / 16: 1.5 % / 0.3 % faster)
static constexpr int PK_TILE = PK_THREADS * PK_ITEMS;          // 4096
static constexpr int RUN_MAX = 64;
static constexpr int LB = 4;                                  // look-back words loaded per round trip

static constexpr uint32_t PK_FLAG_AGG = 1u << 30;
static constexpr uint32_t PK_FLAG_INC = 2u << 30;
static constexpr uint32_t PK_FLAG_MASK = 3u << 30;

enum { CTL_KMIN = 0, CTL_KMAX = 1, CTL_LONGRUN = 2 };

// how the keys are packed, derived by every kernel from (n, kmin, kmax)
struct Packing {
    uint64_t kmin;
    int idx_bits, key_bits, sort_bits, s, up;      // key bits kept / sorted by the passes; right or left shift of key - kmin
    __host__ __device__ uint64_t key_part(uint64_t key) const { return ((key - kmin) >> s) << up; }
    __host__ __device__ int low_bits() const { return key_bits - sort_bits; }      // kept but not sorted: resolved in the runs
};

// bits the passes sort: about log2 n, whole digits, at least two of them
__host__ __device__ inline int sort_bits_of(int ib, int key_bits)
{
    int sb = ((ib + 7) / 8) * 8;
    if (sb < 16) sb = 16;
    return sb < key_bits ? sb : (key_bits / 8) * 8;
}

__device__ __forceinline__ Packing packing_of(uint32_t n, const uint64_t* __restrict__ ctl)
{
    Packing p;
    p.kmin = ~ctl[CTL_KMIN];                                   // kept complemented so that zero-fill initialises it
    const uint64_t span = ctl[CTL_KMAX] - p.kmin;
    int ib = 32 - __clz(n - 1u);                               // bits needed for 0 .. n-1 (n >= 2)
    if (n < 2) ib = 1;
    p.idx_bits = ib < 24 ? 24 : ib;
    p.key_bits = PK_KEYBITS_MAX < 64 - p.idx_bits ? PK_KEYBITS_MAX : 64 - p.idx_bits;      // what fits beside the index
    p.sort_bits = sort_bits_of(ib, p.key_bits);
    const int span_bits = 64 - __clzll((long long)span);       // 0 when all keys are equal
    p.s = span_bits > p.key_bits ? span_bits - p.key_bits : 0;
    p.up = span_bits < p.key_bits ? p.key_bits - span_bits : 0;
    return p;
}

// lanes of the warp holding the same 8-bit digit, from eight ballots (the hardware match.any
// instruction is far slower than this on sm_100)
__device__ __forceinline__ unsigned match_digit(uint32_t d)
{
    unsigned peers = 0xffffffffu;
#pragma unroll
    for (int bit = 0; bit < 8; ++bit) {
        const unsigned mask = (unsigned)((int)(d << (31 - bit)) >> 31);     // all ones if the bit is set
        const unsigned m = __ballot_sync(0xffffffffu, mask != 0u);
        peers &= ~(m ^ mask);                                              // m if set, ~m if not
    }
    return peers;
}

// ---- key range ----------------------------------------------------------------------------------
// (also zeroes the look-back words of the digit passes, which run later: one memset fewer per sort)
__global__ void __launch_bounds__(512) sort_minmax_kernel(const uint64_t* __restrict__ keys, uint64_t n,
                                                          unsigned long long* __restrict__ ctl,
                                                          uint4* __restrict__ lookback4, uint64_t nlookback4)
{
    __shared__ unsigned long long smin[16], smax[16];
    unsigned long long lo = ~0ull, hi = 0ull;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nlookback4; i += stride) lookback4[i] = make_uint4(0u, 0u, 0u, 0u);
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const unsigned long long k = __ldg(keys + i);
        lo = k < lo ? k : lo;
        hi = k > hi ? k : hi;
    }
    for (int d = 16; d > 0; d >>= 1) {
        const unsigned long long a = __shfl_xor_sync(0xffffffffu, lo, d), b = __shfl_xor_sync(0xffffffffu, hi, d);
        lo = a < lo ? a : lo;
        hi = b > hi ? b : hi;
    }
    if ((threadIdx.x & 31) == 0) { smin[threadIdx.x >> 5] = lo; smax[threadIdx.x >> 5] = hi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 16; ++w) { lo = smin[w] < lo ? smin[w] : lo; hi = smax[w] > hi ? smax[w] : hi; }
        atomicMax(ctl + CTL_KMIN, ~lo);
        atomicMax(ctl + CTL_KMAX, hi);
    }
}

// ---- 64-byte star records -------------------------------------------------------------------------
// record i = { r_i, cols[0][i], ..., cols[ncols-1][i], (uint32) id_i, padding }, ncols <= PK_REC_COLS
static constexpr int PK_REC_COLS = 6;

struct PkCols {
    const double* in[HMC_MAX_COLS];
    double* out[HMC_MAX_COLS];
    const uint32_t* id_in;
    uint32_t* id_out;
    int ncols;
};

// Records of the 32 stars base .. base+31 (< n), written by one warp.  Lane l owns slot l & 7 (its source
// array is chosen once) and, in each of 8 steps, star 4*step + (l >> 3): every load instruction reads one
// full sector from each array, every store instruction writes 256 contiguous bytes.
__device__ __forceinline__ void write_records_32(const double* __restrict__ r, const PkCols& g, double* __restrict__ rec,
                                                 uint32_t base, uint32_t n, uint32_t lane)
{
    const uint32_t slot = lane & 7, sub = lane >> 3;
    const double* src = nullptr;
    if (slot == 0) src = r;
    else if ((int)slot <= g.ncols) src = g.in[slot - 1];
    const uint32_t* src_id = ((int)slot == g.ncols + 1) ? g.id_in : nullptr;
    double v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const uint32_t i = base + 4 * j + sub;
        v[j] = 0.0;
        if (i < n) {
            if (src) v[j] = __ldcs(src + i);
            else if (src_id) v[j] = __longlong_as_double((long long)(unsigned long long)__ldcs(src_id + i));
        }
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const uint32_t i = base + 4 * j + sub;
        if (i < n) __stcs(rec + (size_t)i * 8 + slot, v[j]);
    }
}

// ---- digit histograms of the key part, all passes in one read -------------------------------------
static constexpr int PKH_THREADS = 512;
static constexpr int PKH_COPIES = 4;
static constexpr int PKH_UNROLL = 4;

__global__ void __launch_bounds__(PKH_THREADS) sort_pk_histogram_kernel(const uint64_t* __restrict__ keys, uint32_t n,
                                                                        const uint64_t* __restrict__ ctl,
                                                                        uint32_t* __restrict__ hist /*[5][256]*/, PkCols g,
                                                                        double* __restrict__ rec /* nullptr: no records */)
{
    __shared__ uint32_t sh[PKH_COPIES][PK_MAXPASS * PK_RADIX];
    for (int i = threadIdx.x; i < PKH_COPIES * PK_MAXPASS * PK_RADIX; i += PKH_THREADS) (&sh[0][0])[i] = 0;
    __syncthreads();
    const Packing pk = packing_of(n, ctl);
    uint32_t* mine = sh[(threadIdx.x >> 5) % PKH_COPIES];
    const int npass = pk.sort_bits / 8;                         // digits beyond are not sorted
    const int low = pk.low_bits();
    const uint32_t stride = gridDim.x * PKH_THREADS;
    const uint32_t iters = (n + stride - 1) / stride;           // same trip count for every thread
    uint32_t i = blockIdx.x * PKH_THREADS + threadIdx.x;
    for (uint32_t it = 0; it < iters; it += PKH_UNROLL) {
        uint64_t kp[PKH_UNROLL];
        bool ok[PKH_UNROLL];
#pragma unroll
        for (int u = 0; u < PKH_UNROLL; ++u) {                  // all loads first: several keys in flight per thread
            const uint32_t iu = i + u * stride;
            ok[u] = (it + u < iters) && iu < n;
            kp[u] = ok[u] ? __ldcs(keys + iu) : 0ull;
        }
        // the star records of the same stars (this kernel waits on shared-memory atomics and leaves the
        // memory system idle; a warp's 32 keys of one round are 32 consecutive stars)
        if (rec) {
            const uint32_t lane = threadIdx.x & 31;
            for (int u = 0; u < PKH_UNROLL; ++u) {
                const uint32_t base = i + u * stride - lane;
                if (it + u < iters && base < n) write_records_32(reinterpret_cast<const double*>(keys), g, rec, base, n, lane);
            }
        }
#pragma unroll
        for (int u = 0; u < PKH_UNROLL; ++u) {
            if (it + u >= iters) break;                         // uniform over the warp
            const uint64_t k = pk.key_part(kp[u]) >> low;
            if (ok[u]) {
#pragma unroll
                for (int p = 0; p < PK_MAXPASS - 1; ++p)
                    if (p < npass - 1) atomicAdd(&mine[p * PK_RADIX + ((uint32_t)(k >> (8 * p)) & 255u)], 1u);
            }
            // the leading digit takes few distinct values: aggregate across the warp first
            const unsigned live = __ballot_sync(0xffffffffu, ok[u]);
            {
                const int p = npass - 1;
                const uint32_t d = (uint32_t)(k >> (8 * p)) & 255u;
                const unsigned peers = match_digit(d) & live;
                if (ok[u] && (peers & lanemask_lt()) == 0) atomicAdd(&mine[p * PK_RADIX + d], (uint32_t)__popc(peers));
            }
        }
        i += PKH_UNROLL * stride;
    }
    // digits beyond the sorted bits: their passes are never launched; mark them dead (one bin holds every star)
    if (blockIdx.x == 0 && threadIdx.x < PK_MAXPASS && (int)threadIdx.x >= npass) atomicAdd(&hist[threadIdx.x * PK_RADIX], n);
    __syncthreads();
    for (int b = threadIdx.x; b < PK_MAXPASS * PK_RADIX; b += PKH_THREADS) {
        uint32_t c = 0;
#pragma unroll
        for (int q = 0; q < PKH_COPIES; ++q) c += sh[q][b];
        if (c) atomicAdd(&hist[b], c);
    }
}

// exclusive scan of each pass's 256 counts; pass_live[p] = 0 when one bin holds every star
__global__ void sort_pk_scan_hist_kernel(uint32_t* __restrict__ hist, uint32_t n, uint32_t* __restrict__ pass_live)
{
    __shared__ uint32_t sh[PK_RADIX];
    const int p = blockIdx.x, d = threadIdx.x;
    const uint32_t c = hist[p * PK_RADIX + d];
    sh[d] = c;
    __syncthreads();
    for (int off = 1; off < PK_RADIX; off <<= 1) {
        const uint32_t v = (d >= off) ? sh[d - off] : 0;
        __syncthreads();
        sh[d] += v;
        __syncthreads();
    }
    hist[p * PK_RADIX + d] = sh[d] - c;
    const int single = __syncthreads_or(c == n);
    if (d == 0) pass_live[p] = single ? 0u : 1u;
}

// ---- one digit pass over the packed words -------------------------------------------------------
// Same scheme as the general sort (tiles in ticket order, stable warp-level ranking, decoupled
// look-back over per-tile digit counts, scatter through shared memory), but 8 bytes per star.
struct PkSmem {
    uint64_t words[PK_TILE];                       // 32 KB
    uint32_t warp_counts[PK_WARPS][PK_RADIX];      // 16 KB
    uint32_t digit_base[PK_RADIX];
    uint32_t global_base[PK_RADIX];
    uint32_t tile;
};

struct PkBuffers {
    const uint64_t* keys_src;      // the caller's r_in (read by the first live pass)
    uint64_t* buf[2];              // live pass number i writes buf[i & 1]
};

__global__ void __launch_bounds__(PK_THREADS, 2)
sort_pk_pass_kernel(PkBuffers b, uint32_t n, const uint64_t* __restrict__ ctl,
                    const uint32_t* __restrict__ bin_offset /*[256] exclusive*/, uint32_t* __restrict__ lookback,
                    uint32_t* __restrict__ ticket, const uint32_t* __restrict__ pass_live, int pass)
{
    if (!pass_live[pass]) return;
    int live_before = 0;
    for (int p = 0; p < pass; ++p) live_before += pass_live[p] ? 1 : 0;
    const bool first = live_before == 0;
    const uint64_t* __restrict__ in = b.buf[(live_before & 1) ^ 1];
    uint64_t* __restrict__ out = b.buf[live_before & 1];
    const Packing pk = packing_of(n, ctl);
    const int shift = pk.idx_bits + pk.low_bits() + 8 * pass;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    PkSmem& s = *reinterpret_cast<PkSmem*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tiles = (n + PK_TILE - 1) / PK_TILE;
    for (;;) {                                                  // persistent CTAs: tiles in ticket order
    __syncthreads();                                            // previous tile's shared memory is no longer read
    if (tid == 0) s.tile = atomicAdd(ticket, 1u);
    for (int i = tid; i < PK_WARPS * PK_RADIX; i += PK_THREADS) (&s.warp_counts[0][0])[i] = 0;
    __syncthreads();
    const uint32_t tile = s.tile;
    if (tile >= tiles) break;
    const uint32_t tile_base = tile * PK_TILE;
    const uint32_t valid = min((uint32_t)PK_TILE, n - tile_base);
    // load, warp-striped: item i of lane l sits at tile position warp*256 + i*32 + l
    uint64_t w[PK_ITEMS];
    const uint32_t wbase = warp * (32 * PK_ITEMS) + lane;
#pragma unroll
    for (int i = 0; i < PK_ITEMS; ++i) {
        const uint32_t pos = wbase + i * 32;
        if (pos < valid) {
            const uint32_t g = tile_base + pos;
            w[i] = first ? ((pk.key_part(__ldcs(b.keys_src + g)) << pk.idx_bits) | g) : __ldcs(in + g);
        } else w[i] = ~0ull;                                    // padding: the largest digit of the pass, ranks last in the tile
    }
    // stable rank inside the warp, item by item
    uint32_t rank[PK_ITEMS];
    uint32_t* wc = s.warp_counts[warp];
#pragma unroll
    for (int i = 0; i < PK_ITEMS; ++i) {
        const uint32_t d = (uint32_t)(w[i] >> shift) & 255u;
        const unsigned peers = match_digit(d);
        const int leader = __ffs(peers) - 1;
        uint32_t before = 0;
        if (lane == leader) { before = wc[d]; wc[d] = before + __popc(peers); }
        before = __shfl_sync(0xffffffffu, before, leader);
        rank[i] = before + __popc(peers & lanemask_lt());
        __syncwarp();
    }
    __syncthreads();
    // digit d is owned by thread d: its count in the tile is published at once (the later tiles' look-back
    // needs it), the look-back itself is left until after the scatter so that the earlier tiles have had time
    // to publish their inclusive sums (shorter chains)
    uint32_t count = 0;
    if (tid < PK_RADIX) {
        const int d = tid;
        uint32_t run = 0;
#pragma unroll
        for (int q = 0; q < PK_WARPS; ++q) { const uint32_t c = s.warp_counts[q][d]; s.warp_counts[q][d] = run; run += c; }
        count = run;
        // padding is not data.  Its digit is 255 except in a last pass whose digit reaches beyond bit 63
        // (n > 2^24: the index takes more than 24 bits), where the bits above the word read as zero.
        if (d == (int)((uint32_t)(~0ull >> shift) & 255u)) count -= (PK_TILE - valid);
        st_volatile_u32(lookback + (size_t)tile * PK_RADIX + d, PK_FLAG_AGG | count);
        s.digit_base[d] = run;                                  // padded tile count, scanned below
    }
    __syncthreads();
    // exclusive scan of the 256 tile counts by warp 0 (8 per lane)
    if (warp == 0) {
        uint32_t c[8], sum = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) { c[i] = s.digit_base[lane * 8 + i]; sum += c[i]; }
        uint32_t inc = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
        uint32_t run = inc - sum;
#pragma unroll
        for (int i = 0; i < 8; ++i) { s.digit_base[lane * 8 + i] = run; run += c[i]; }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < PK_ITEMS; ++i) {
        const uint32_t d = (uint32_t)(w[i] >> shift) & 255u;
        s.words[s.digit_base[d] + s.warp_counts[warp][d] + rank[i]] = w[i];
    }
    if (tid < PK_RADIX) {
        const int d = tid;
        uint32_t* my = lookback + (size_t)tile * PK_RADIX + d;
        // look back LB tiles at a time (their words are loaded together: one L2 round trip for LB steps)
        uint32_t excl = 0;
        for (int64_t t = (int64_t)tile - 1; t >= 0; t -= LB) {
            uint32_t v[LB];
#pragma unroll
            for (int j = 0; j < LB; ++j) v[j] = (t - j >= 0) ? ld_volatile_u32(lookback + (size_t)(t - j) * PK_RADIX + d) : PK_FLAG_INC;
            bool stop = false;
#pragma unroll
            for (int j = 0; j < LB; ++j) {
                if (stop) break;
                uint32_t x = v[j];
                while ((x & PK_FLAG_MASK) == 0) x = ld_volatile_u32(lookback + (size_t)(t - j) * PK_RADIX + d);
                excl += x & ~PK_FLAG_MASK;
                stop = (x & PK_FLAG_MASK) == PK_FLAG_INC;
            }
            if (stop) break;
        }
        st_volatile_u32(my, PK_FLAG_INC | (excl + count));
        s.global_base[d] = bin_offset[d] + excl - s.digit_base[d];   // global position = global_base[d] + tile position
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < PK_ITEMS; ++i) {
        const uint32_t pos = tid + i * PK_THREADS;
        if (pos < valid) {
            const uint64_t v = s.words[pos];
            out[s.global_base[(uint32_t)(v >> shift) & 255u] + pos] = v;
        }
    }
    }   // tile loop
}

// ---- final kernel: resolve runs, move the records ---------------------------------------------------
// Each warp takes 32 consecutive output positions.  The owner lane of a position finds the
// star's index and its place (run resolution); then the records are fetched by lane PAIRS, the
// two 32-byte halves of a record in one load instruction, so that a record costs one 64-byte DRAM
// fetch (two separate loads were seen to fetch 64 bytes each), and each half is stored by the
// lane that loaded it.
template <bool USE_REC>
__global__ void __launch_bounds__(256)
sort_pk_finish_kernel(PkBuffers b, const double* __restrict__ rec, PkCols g, uint32_t n, uint64_t* __restrict__ ctl,
                      const uint32_t* __restrict__ pass_live, double* __restrict__ r_sorted, uint32_t* __restrict__ perm)
{
    int live = 0;
    for (int p = 0; p < PK_MAXPASS; ++p) live += pass_live[p] ? 1 : 0;
    const uint64_t* __restrict__ fin = b.buf[(live - 1) & 1];
    const Packing pk = packing_of(n, ctl);
    const int ib = pk.idx_bits;
    const uint64_t idx_mask = (1ull << ib) - 1;
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t stride = gridDim.x * blockDim.x;
    const uint32_t rounds = (n + stride - 1) / stride;                     // whole warps stay together
    uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    for (uint32_t it = 0; it < rounds; ++it, k += stride) {
        const bool in = k < n;
        uint32_t idx = 0, dest = k;
        if (in) {
            const uint64_t w = live ? __ldg(fin + k) : (uint64_t)k;        // no live pass: every key part equal
            idx = (uint32_t)(w & idx_mask);
            const int low = pk.low_bits();
            if (live && (low > 0 || pk.s > 0)) {                           // else equal sorted bits are equal keys, in input order
                const int rs = ib + low;                                   // the passes sorted the bits from rs up
                const uint64_t sk = w >> rs;
                const bool eq_l = k > 0 && (__ldg(fin + k - 1) >> rs) == sk;
                const bool eq_r = k + 1 < n && (__ldg(fin + k + 1) >> rs) == sk;
                if (eq_l || eq_r) {                                        // member of a run: rank inside it by (key, index)
                    uint32_t a = k, e = k + 1;
                    while (a > 0 && k - a <= RUN_MAX && (__ldg(fin + a - 1) >> rs) == sk) --a;
                    while (e < n && e - a <= RUN_MAX + 1 && (__ldg(fin + e) >> rs) == sk) ++e;
                    if (e - a > RUN_MAX) ctl[CTL_LONGRUN] = 1;            // the general sort redoes the call
                    else {
                        const uint64_t kept = w >> ib;
                        uint64_t mine = 0;
                        bool have_mine = false;
                        uint32_t below = 0;
                        for (uint32_t j = a; j < e; ++j) {
                            if (j == k) continue;
                            const uint64_t wj = __ldg(fin + j);
                            bool less = wj < w;                            // other kept key bits, or the same and a lower index
                            if (pk.s > 0 && (wj >> ib) == kept) {          // all kept bits agree but bits were dropped: full keys
                                if (!have_mine) { mine = __ldg(b.keys_src + idx); have_mine = true; }
                                const uint64_t other = __ldg(b.keys_src + (uint32_t)(wj & idx_mask));
                                less = other < mine || (other == mine && wj < w);
                            }
                            below += less ? 1u : 0u;
                        }
                        dest = a + below;
                    }
                }
            }
            __stcs(perm + dest, idx);
        }
        if (USE_REC) {
            const int h = lane & 1;
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const int src = t * 16 + (lane >> 1);
                const uint32_t idx_j = __shfl_sync(0xffffffffu, idx, src);
                const uint32_t dest_j = __shfl_sync(0xffffffffu, dest, src);
                const bool in_j = __shfl_sync(0xffffffffu, (int)in, src) != 0;
                if (in_j) {
                    double v[4];
                    const double* p = rec + (size_t)idx_j * 8 + h * 4;
                    asm("ld.global.nc.L1::no_allocate.L2::64B.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v[0]), "=d"(v[1]), "=d"(v[2]), "=d"(v[3]) : "l"(p));
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int slot = h * 4 + q;
                        if (slot == 0) __stcs(r_sorted + dest_j, v[q]);
                        else if (slot <= g.ncols) __stcs(g.out[slot - 1] + dest_j, v[q]);
                        else if (slot == g.ncols + 1 && g.id_out)
                            __stcs(g.id_out + dest_j, (uint32_t)(unsigned long long)__double_as_longlong(v[q]));
                    }
                }
            }
        } else if (in) {
            __stcs(r_sorted + dest, __longlong_as_double((long long)__ldg(b.keys_src + idx)));
#pragma unroll
            for (int c = 0; c < HMC_MAX_COLS; ++c)
                if (c < g.ncols) __stcs(g.out[c] + dest, __ldg(g.in[c] + idx));
            if (g.id_out) __stcs(g.id_out + dest, __ldg(g.id_in + idx));
        }
    }
}

// ---- host side ----------------------------------------------------------------------------------------
// Enqueues the fast path.  The caller then enqueues the general sort guarded by ctl[CTL_LONGRUN].
hmc_status sort_fast(uint64_t n, const double* r_in, double* r_sorted, uint32_t* perm, int ncols,
                     const double* const* cols_in, double* const* cols_out, const uint32_t* id_in, uint32_t* id_out,
                     const Workspace& ws, cudaStream_t st)
{
    const uint32_t tiles = (uint32_t)((n + PK_TILE - 1) / PK_TILE);
    const int sms = sm_count();
    const uint64_t* keys = reinterpret_cast<const uint64_t*>(r_in);
    uint32_t* pass_live = ws.pk_tickets + 8;
    // sortctl, pk_hist and pk_tickets are adjacent in the workspace: one memset
    HMC_CUDA_TRY(cudaMemsetAsync(ws.sortctl, 0, reinterpret_cast<char*>(ws.pk_tickets + 16) - reinterpret_cast<char*>(ws.sortctl), st));
    PkCols g{};
    g.ncols = ncols;
    for (int c = 0; c < ncols; ++c) { g.in[c] = cols_in[c]; g.out[c] = cols_out[c]; }
    g.id_in = id_in; g.id_out = id_out;
    const bool use_rec = (ncols > 0 || id_in) && ncols <= PK_REC_COLS;
    const int stream_blocks = (int)umin64((n + 511) / 512, (uint64_t)sms * 4);
    int ib = 1;
    while ((1ull << ib) < n) ++ib;                                          // as packing_of
    const int idx_bits = ib < 24 ? 24 : ib;
    const int key_bits = PK_KEYBITS_MAX < 64 - idx_bits ? PK_KEYBITS_MAX : 64 - idx_bits;
    const int npass = sort_bits_of(ib, key_bits) / 8;                       // digits of the leading bits only
    sort_minmax_kernel<<<stream_blocks, 512, 0, st>>>(keys, n, reinterpret_cast<unsigned long long*>(ws.sortctl),
                                                      reinterpret_cast<uint4*>(ws.lookback), (uint64_t)npass * tiles * PK_RADIX / 4);
    HMC_LAUNCH_CHECK();
    sort_pk_histogram_kernel<<<(int)umin64((n + PKH_THREADS - 1) / PKH_THREADS, (uint64_t)sms * 3), PKH_THREADS, 0, st>>>(
        keys, (uint32_t)n, ws.sortctl, ws.pk_hist, g, use_rec ? reinterpret_cast<double*>(ws.rec) : nullptr);
    HMC_LAUNCH_CHECK();
    sort_pk_scan_hist_kernel<<<PK_MAXPASS, PK_RADIX, 0, st>>>(ws.pk_hist, (uint32_t)n, pass_live);
    HMC_LAUNCH_CHECK();
    const int copy_blocks = (int)umin64((n + 255) / 256, (uint64_t)sms * 8);
    static std::atomic<uint64_t> opted{ 0 };
    hmc_status so = smem_opt_in(opted, sort_pk_pass_kernel, sizeof(PkSmem));
    if (so != HMC_OK) return so;
    PkBuffers b{ keys, { ws.keys_alt, ws.pk_alt } };
    for (int p = 0; p < npass; ++p) {
        sort_pk_pass_kernel<<<(int)umin64(tiles, (uint64_t)sms * 2), PK_THREADS, sizeof(PkSmem), st>>>(b, (uint32_t)n, ws.sortctl, ws.pk_hist + p * PK_RADIX,
                                                                       ws.lookback + (size_t)p * tiles * PK_RADIX,
                                                                       ws.pk_tickets + p, pass_live, p);
        HMC_LAUNCH_CHECK();
    }
    if (use_rec)
        sort_pk_finish_kernel<true><<<copy_blocks, 256, 0, st>>>(b, reinterpret_cast<const double*>(ws.rec), g, (uint32_t)n,
                                                                 ws.sortctl, pass_live, r_sorted, perm);
    else
        sort_pk_finish_kernel<false><<<copy_blocks, 256, 0, st>>>(b, nullptr, g, (uint32_t)n, ws.sortctl, pass_live, r_sorted, perm);
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

}  // namespace hmc
