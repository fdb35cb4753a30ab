// hmc_potential.cu -- S2: Phi_k = -G (M_k / r_k + S_k) on the radius-sorted arrays.
//
// The paper computes Phi by the backward recursion Eq. 2-5 and calls it "inherently sequential"
// (PAPER.md:185).  Here the stars are cut into CHUNKS of consecutive tiles (a tile = 2048 stars), one chunk per
// CTA of a grid that fills the machine once, and the stage is two launches without any inter-CTA waiting:
//   1. potential_reduce_kernel : every warp sums slices of 1024 consecutive stars, T_m = sum m_i and
//                                T_t = sum fl(m_i / r_i); per-slice and per-chunk totals go to the workspace.
//   2. potential_apply_kernel  : the CTA of chunk c adds up the chunk totals before (T_m) and after (T_t) its
//                                chunk -- a few hundred values, once per CTA -- and the slice totals inside it,
//                                then walks its tiles from the last to the first: forward scan of m and
//                                backward scan of m/r in registers, M_k and S_k rounded once,
//                                Phi_k = -(G*(M_k/r_k + S_k)).
// (Round 1 had a third, single-CTA launch between the two that scanned ~5000 tile totals while the rest of the
// GPU idled for 20 us.)  The reduce launch walks each chunk forwards, the apply launch backwards, so the tail of
// every chunk is still in the 126 MB L2 when it is read the second time.
//
// Every partial sum is double-double (106 bits), so M_k and S_k are the exact sums rounded once and do not
// depend on the association order (R1p).  Adding two double-double PARTIAL SUMS uses the short form of
// the addition (one two_sum and a renormalisation): its error bound, 2^-104 relative to |a| + |b|, is relative to
// the result because the summands m_i and m_i / r_i are non-negative (precondition m >= 0, r > 0).
#include "hmc_common.cuh"

namespace hmc {

static constexpr int SCAN_THREADS = 256;
static constexpr int SCAN_WARPS = SCAN_THREADS / 32;
static constexpr int SCAN_ITEMS = SCAN_TILE / SCAN_THREADS;   // 8 consecutive stars per thread in the apply launch
static constexpr int SLICE = 1024;                            // stars per warp-slice of the reduce launch
static constexpr int SLICES_PER_TILE = SCAN_TILE / SLICE;     // 2
static constexpr int CHUNK_CTAS_PER_SM = 3;                   // chunks = CTAs resident at once: 80 registers x 256 threads (2 and 4 measured slower)
static constexpr int RED_BATCH = 4;                           // 16-byte loads in flight per array and lane in the reduce launch (2, 8, 16: no better)
static_assert(SCAN_ITEMS == 8, "the apply launch loads 2 x 4 consecutive doubles per thread and array");

// double-double sum of two double-double values of the same sign (see the header): 11 operations instead of 20
__device__ __forceinline__ dd dd_add_pos(dd a, dd b)
{
    dd s = two_sum(a.hi, b.hi);
    s.lo += a.lo + b.lo;
    return quick_two_sum(s.hi, s.lo);
}

__device__ __forceinline__ dd dd_shfl_xor(dd v, int mask)
{
    return dd{ __shfl_xor_sync(0xffffffffu, v.hi, mask), __shfl_xor_sync(0xffffffffu, v.lo, mask) };
}
__device__ __forceinline__ dd dd_shfl_down(dd v, int delta)
{
    return dd{ __shfl_down_sync(0xffffffffu, v.hi, delta), __shfl_down_sync(0xffffffffu, v.lo, delta) };
}
__device__ __forceinline__ dd dd_shfl(dd v, int lane)
{
    return dd{ __shfl_sync(0xffffffffu, v.hi, lane), __shfl_sync(0xffffffffu, v.lo, lane) };
}

__device__ __forceinline__ void ld4(const double* __restrict__ p, double v[4])
{
    asm("ld.global.nc.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v[0]), "=d"(v[1]), "=d"(v[2]), "=d"(v[3]) : "l"(p));
}
__device__ __forceinline__ void st4(double* __restrict__ p, const double v[4])
{
    asm volatile("st.global.cs.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(v[0]), "d"(v[1]), "d"(v[2]), "d"(v[3]) : "memory");
}

// How the stars are cut up; the same for both launches.  Chunk c = tiles [c * tpc, min(ntiles, (c+1) * tpc)).
struct ScanPlan {
    uint32_t ntiles, nslices, tpc, nchunks;
};

// Tiles per chunk whose offsets fit the apply launch's shared arrays.  One chunk per resident CTA would need 296 at
// n = HMC_MAX_N on 148 SMs (and more on a smaller GPU): scan_plan caps tpc here and lets the grid grow beyond one
// wave instead -- no CTA of either launch waits for another, so any number of chunks is correct, and the workspace
// has room for one chunk total per tile.
static constexpr int MAX_TPC_SMEM = 256;

static inline ScanPlan scan_plan(uint64_t n, int sms)
{
    ScanPlan p;
    p.ntiles = (uint32_t)((n + SCAN_TILE - 1) / SCAN_TILE);
    p.nslices = (uint32_t)((n + SLICE - 1) / SLICE);
    const uint32_t want = (uint32_t)sms * CHUNK_CTAS_PER_SM;
    p.tpc = (p.ntiles + want - 1) / want;
    if (p.tpc == 0) p.tpc = 1;
    if (p.tpc > (uint32_t)MAX_TPC_SMEM) p.tpc = MAX_TPC_SMEM;
    p.nchunks = (p.ntiles + p.tpc - 1) / p.tpc;
    return p;
}

// ---- 1. slice and chunk totals -----------------------------------------------------------------
// slice_tot[s] = (T_m.hi, T_m.lo, T_t.hi, T_t.lo) of stars [s * 1024, (s+1) * 1024); chunk_tot[c] likewise for
// the whole chunk.  The order of the elements inside a slice is irrelevant for a sum, so the loads are fully
// coalesced 16-byte loads; a warp works alone (no barrier inside the loop).
__global__ void __launch_bounds__(SCAN_THREADS, CHUNK_CTAS_PER_SM)
potential_reduce_kernel(const double* __restrict__ r, const double* __restrict__ m, uint64_t n, ScanPlan plan,
                        double4* __restrict__ slice_tot, double4* __restrict__ chunk_tot)
{
    __shared__ dd sm_m[SCAN_WARPS], sm_t[SCAN_WARPS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t c = blockIdx.x;
    const uint32_t s0 = c * plan.tpc * SLICES_PER_TILE;
    const uint32_t s1 = min(plan.nslices, (c + 1) * plan.tpc * SLICES_PER_TILE);
    const bool aligned = ((reinterpret_cast<uintptr_t>(r) | reinterpret_cast<uintptr_t>(m)) & 15) == 0;
    dd cm{ 0.0, 0.0 }, ct{ 0.0, 0.0 };                           // this warp's share of the chunk
    for (uint32_t s = s0 + warp; s < s1; s += SCAN_WARPS) {
        const uint64_t base = (uint64_t)s * SLICE;
        dd am{ 0.0, 0.0 }, at{ 0.0, 0.0 }, bm{ 0.0, 0.0 }, bt{ 0.0, 0.0 };   // two chains per sum: the adds are dependent
        if (base + SLICE <= n && aligned) {
            const double2* r2 = reinterpret_cast<const double2*>(r + base) + lane;
            const double2* m2 = reinterpret_cast<const double2*>(m + base) + lane;
#pragma unroll
            for (int h = 0; h < 16 / RED_BATCH; ++h) {
                double2 rv[RED_BATCH], mv[RED_BATCH];
#pragma unroll
                for (int i = 0; i < RED_BATCH; ++i) { rv[i] = __ldg(r2 + (h * RED_BATCH + i) * 32); mv[i] = __ldg(m2 + (h * RED_BATCH + i) * 32); }
#pragma unroll
                for (int i = 0; i < RED_BATCH; ++i) {
                    am = dd_add_d(am, mv[i].x); bm = dd_add_d(bm, mv[i].y);
                    at = dd_add_d(at, mv[i].x / rv[i].x); bt = dd_add_d(bt, mv[i].y / rv[i].y);
                }
            }
            am = dd_add_pos(am, bm); at = dd_add_pos(at, bt);
        } else {
            for (int i = 0; i < SLICE / 32; ++i) {
                const uint64_t a = base + (uint64_t)i * 32 + lane;
                if (a < n) { const double mm = m[a]; am = dd_add_d(am, mm); at = dd_add_d(at, mm / r[a]); }
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) { am = dd_add_pos(am, dd_shfl_xor(am, d)); at = dd_add_pos(at, dd_shfl_xor(at, d)); }
        if (lane == 0) slice_tot[s] = make_double4(am.hi, am.lo, at.hi, at.lo);
        cm = dd_add_pos(cm, am); ct = dd_add_pos(ct, at);         // the same value in every lane
    }
    if (lane == 0) { sm_m[warp] = cm; sm_t[warp] = ct; }
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int w = 1; w < SCAN_WARPS; ++w) { cm = dd_add_pos(cm, sm_m[w]); ct = dd_add_pos(ct, sm_t[w]); }
        chunk_tot[c] = make_double4(cm.hi, cm.lo, ct.hi, ct.lo);
    }
}

// ---- 2. per-tile scans and Phi -----------------------------------------------------------------
// Sharded step: further destinations of the shard's slice of the replicated table, e.g. the other
// GPUs' copies at this shard's offset, reached by peer access over NVLink.  The launch that produces Phi and M stores
// them (and the radii it has in registers) there tile by tile, so the table's all-gather is done when the scan is.
struct PushTargets {
    int npeers;
    double* r[HMC_MAX_PEERS];
    double* phi[HMC_MAX_PEERS];
    double* m_cum[HMC_MAX_PEERS];
};

__global__ void __launch_bounds__(SCAN_THREADS, CHUNK_CTAS_PER_SM)
potential_apply_kernel(const double* __restrict__ r, const double* __restrict__ m, double* __restrict__ phi,
                       double* __restrict__ m_cum, uint64_t n, double G, ScanPlan plan,
                       const double4* __restrict__ slice_tot, const double4* __restrict__ chunk_tot,
                       const double4* __restrict__ ext_tot, uint32_t nranks, uint32_t rank, PushTargets push)
{
    __shared__ dd sm_m[2][SCAN_WARPS], sm_t[2][SCAN_WARPS];     // per-warp totals of the tile being scanned (by tile parity)
    __shared__ dd sm_pm[MAX_TPC_SMEM];                          // sum of m over everything before tile k of this chunk
    __shared__ dd sm_slice[MAX_TPC_SMEM * SLICES_PER_TILE];     // T_m of the chunk's slices (prologue only)
    __shared__ dd sm_after[2];                                  // sum of m/r over everything after the current tile (by parity)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t c = blockIdx.x;
    const uint32_t t0 = c * plan.tpc, t1 = min(plan.ntiles, t0 + plan.tpc);

    // ---- prologue: what lies before and after this chunk, from the chunk totals (once per CTA)
    {
        dd pm{ 0.0, 0.0 }, st{ 0.0, 0.0 };
        for (uint32_t j = tid; j < plan.nchunks; j += SCAN_THREADS) {
            if (j == c) continue;
            const double4 v = chunk_tot[j];
            if (j < c) pm = dd_add_pos(pm, dd{ v.x, v.y });
            else st = dd_add_pos(st, dd{ v.z, v.w });
        }
        // sharded step: the other shards of the cluster lie wholly before (lower rank) or after (higher rank) this one
        for (uint32_t j = tid; ext_tot != nullptr && j < nranks; j += SCAN_THREADS) {
            if (j == rank) continue;
            const double4 v = ext_tot[j];
            if (j < rank) pm = dd_add_pos(pm, dd{ v.x, v.y });
            else st = dd_add_pos(st, dd{ v.z, v.w });
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) { pm = dd_add_pos(pm, dd_shfl_xor(pm, d)); st = dd_add_pos(st, dd_shfl_xor(st, d)); }
        if (lane == 0) { sm_m[0][warp] = pm; sm_t[0][warp] = st; }
        const uint32_t sl0 = t0 * SLICES_PER_TILE, sl1 = min(plan.nslices, t1 * SLICES_PER_TILE);
        for (uint32_t s = sl0 + tid; s < sl1; s += SCAN_THREADS) { const double4 v = slice_tot[s]; sm_slice[s - sl0] = dd{ v.x, v.y }; }
        __syncthreads();
        if (tid == 0) {
#pragma unroll
            for (int w = 1; w < SCAN_WARPS; ++w) { pm = dd_add_pos(pm, sm_m[0][w]); st = dd_add_pos(st, sm_t[0][w]); }
            sm_after[(t1 - 1) & 1] = st;
            // offsets of the chunk's tiles: the slice totals of the reduce launch, added up in order
            dd run = pm;
            for (uint32_t k = 0; k < t1 - t0; ++k) {
                sm_pm[k] = run;
                for (uint32_t s = k * SLICES_PER_TILE; s < min(sl1 - sl0, (k + 1) * SLICES_PER_TILE); ++s) run = dd_add_pos(run, sm_slice[s]);
            }
        }
        __syncthreads();
    }

    const bool al_in = ((reinterpret_cast<uintptr_t>(r) | reinterpret_cast<uintptr_t>(m)) & 31) == 0;
    const bool al_out = ((reinterpret_cast<uintptr_t>(phi) | reinterpret_cast<uintptr_t>(m_cum)) & 31) == 0;
    for (uint32_t tile = t1; tile-- > t0;) {                      // last tile of the chunk first
        const uint64_t p0 = (uint64_t)tile * SCAN_TILE + (uint64_t)tid * SCAN_ITEMS;
        const bool full = (uint64_t)tile * SCAN_TILE + SCAN_TILE <= n;
        double rr[SCAN_ITEMS], mm[SCAN_ITEMS], tt[SCAN_ITEMS];
        if (full && al_in) {
            ld4(r + p0, rr); ld4(r + p0 + 4, rr + 4);
            ld4(m + p0, mm); ld4(m + p0 + 4, mm + 4);
        } else {
#pragma unroll
            for (int i = 0; i < SCAN_ITEMS; ++i) {
                const uint64_t p = p0 + i;
                rr[i] = (p < n) ? r[p] : 1.0;
                mm[i] = (p < n) ? m[p] : 0.0;
            }
        }
        dd tm{ 0.0, 0.0 }, ts{ 0.0, 0.0 }, um{ 0.0, 0.0 }, us{ 0.0, 0.0 };   // two chains per sum: the adds are dependent
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS; ++i) tt[i] = mm[i] / rr[i];
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS / 2; ++i) {
            tm = dd_add_d(tm, mm[i]); um = dd_add_d(um, mm[i + SCAN_ITEMS / 2]);
            ts = dd_add_d(ts, tt[i]); us = dd_add_d(us, tt[i + SCAN_ITEMS / 2]);
        }
        tm = dd_add_pos(tm, um); ts = dd_add_pos(ts, us);
        dd im = tm, it = ts;                                       // inclusive over lanes: forward m, backward t
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const dd up = dd_shfl_up(im, d);
            if (lane >= d) im = dd_add_pos(up, im);
            const dd dn = dd_shfl_down(it, d);
            if (lane + d < 32) it = dd_add_pos(it, dn);
        }
        const int par = tile & 1;                                  // shared words alternate between two sets: one barrier per tile
        if (lane == 31) sm_m[par][warp] = im;
        if (lane == 0) sm_t[par][warp] = it;
        __syncthreads();
        // everything before this thread's stars (m) / after them (m/r): chunk offset, earlier / later warps, lanes
        dd em = sm_pm[tile - t0], et = sm_after[par];
        if (tid == 0) {                                            // the tile's m/r lies "after" the next (earlier) tile
            dd a = et;
#pragma unroll
            for (int w = 0; w < SCAN_WARPS; ++w) a = dd_add_pos(a, sm_t[par][w]);
            sm_after[par ^ 1] = a;
        }
        for (int w = 0; w < warp; ++w) em = dd_add_pos(em, sm_m[par][w]);
        for (int w = SCAN_WARPS - 1; w > warp; --w) et = dd_add_pos(et, sm_t[par][w]);
        {
            const dd pm = dd_shfl_up(im, 1), pt = dd_shfl_down(it, 1);
            if (lane > 0) em = dd_add_pos(em, pm);
            if (lane < 31) et = dd_add_pos(et, pt);
        }
        double Mk[SCAN_ITEMS], ph[SCAN_ITEMS];
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS; ++i) { em = dd_add_d(em, mm[i]); Mk[i] = em.hi; }      // inclusive prefix, rounded once
#pragma unroll
        for (int i = SCAN_ITEMS - 1; i >= 0; --i) {
            ph[i] = -(G * (Mk[i] / rr[i] + et.hi));                // Eq. 1 at r = r_k; et.hi = S_k, exclusive suffix rounded once
            et = dd_add_d(et, tt[i]);
        }
        if (full && al_out) {
            st4(phi + p0, ph); st4(phi + p0 + 4, ph + 4);
            st4(m_cum + p0, Mk); st4(m_cum + p0 + 4, Mk + 4);
        } else {
#pragma unroll
            for (int i = 0; i < SCAN_ITEMS; ++i) {
                const uint64_t p = p0 + i;
                if (p < n) { phi[p] = ph[i]; m_cum[p] = Mk[i]; }
            }
        }
        for (int g = 0; g < push.npeers; ++g) {                    // the same slice of every peer's table
            double *pr = push.r[g], *pp = push.phi[g], *pc = push.m_cum[g];
            const bool al = ((reinterpret_cast<uintptr_t>(pr) | reinterpret_cast<uintptr_t>(pp) | reinterpret_cast<uintptr_t>(pc)) & 31) == 0;
            if (full && al) {
                st4(pr + p0, rr); st4(pr + p0 + 4, rr + 4);
                st4(pp + p0, ph); st4(pp + p0 + 4, ph + 4);
                st4(pc + p0, Mk); st4(pc + p0 + 4, Mk + 4);
            } else {
#pragma unroll
                for (int i = 0; i < SCAN_ITEMS; ++i) {
                    const uint64_t p = p0 + i;
                    if (p < n) { pr[p] = rr[i]; pp[p] = ph[i]; pc[p] = Mk[i]; }
                }
            }
        }
    }
}

// totals of a whole array (sharded step): the chunk totals of the reduce launch added up by one CTA
__global__ void __launch_bounds__(SCAN_THREADS) potential_sum_chunks_kernel(const double4* __restrict__ chunk_tot, uint32_t nchunks,
                                                                            double4* __restrict__ out)
{
    __shared__ dd sm_m[SCAN_WARPS], sm_t[SCAN_WARPS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    dd am{ 0.0, 0.0 }, at{ 0.0, 0.0 };
    for (uint32_t j = tid; j < nchunks; j += SCAN_THREADS) {
        const double4 v = chunk_tot[j];
        am = dd_add_pos(am, dd{ v.x, v.y }); at = dd_add_pos(at, dd{ v.z, v.w });
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { am = dd_add_pos(am, dd_shfl_xor(am, d)); at = dd_add_pos(at, dd_shfl_xor(at, d)); }
    if (lane == 0) { sm_m[warp] = am; sm_t[warp] = at; }
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int w = 1; w < SCAN_WARPS; ++w) { am = dd_add_pos(am, sm_m[w]); at = dd_add_pos(at, sm_t[w]); }
        *out = make_double4(am.hi, am.lo, at.hi, at.lo);
    }
}

// number of radii <= splitter j, j = 0 .. nsplit-1 (sample sort, phase 4: "the positions of the splitter points in the
// local array are determined by binary search"); one thread per splitter
__global__ void partition_points_kernel(const double* __restrict__ r, uint64_t n, const double* __restrict__ splitters,
                                        uint32_t nsplit, unsigned long long* __restrict__ counts)
{
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nsplit) return;
    const double x = splitters[j];
    uint64_t lo = 0, hi = n;                                     // first position whose radius is > x
    while (lo < hi) {
        const uint64_t mid = lo + (hi - lo) / 2;
        if (r[mid] <= x) lo = mid + 1; else hi = mid;
    }
    counts[j] = lo;
}

hmc_status partition_points(uint64_t n, const double* r_sorted, uint32_t nsplit, const double* splitters, uint64_t* counts,
                            cudaStream_t st)
{
    if (nsplit == 0) return HMC_OK;
    partition_points_kernel<<<(nsplit + 127) / 128, 128, 0, st>>>(r_sorted, n, splitters, nsplit,
                                                                   reinterpret_cast<unsigned long long*>(counts));
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

hmc_status potential_totals(uint64_t n, const double* r, const double* m, double* totals4, const Workspace& ws, cudaStream_t st)
{
    const ScanPlan plan = scan_plan(n, sm_count());
    double4* slice_tot = reinterpret_cast<double4*>(ws.scan_status);
    double4* chunk_tot = slice_tot + plan.nslices;
    if (n > 0) {
        potential_reduce_kernel<<<plan.nchunks, SCAN_THREADS, 0, st>>>(r, m, n, plan, slice_tot, chunk_tot);
        HMC_LAUNCH_CHECK();
    }
    potential_sum_chunks_kernel<<<1, SCAN_THREADS, 0, st>>>(chunk_tot, n > 0 ? plan.nchunks : 0u, reinterpret_cast<double4*>(totals4));
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

hmc_status potential(uint64_t n, double G, const double* r, const double* m, double* phi, double* m_cum,
                     const double* ext_tot, uint32_t nranks, uint32_t rank, const Workspace& ws, cudaStream_t st,
                     int npeers, double* const* peer_r, double* const* peer_phi, double* const* peer_m_cum)
{
    PushTargets push{};
    push.npeers = npeers;
    for (int g = 0; g < npeers; ++g) { push.r[g] = peer_r[g]; push.phi[g] = peer_phi[g]; push.m_cum[g] = peer_m_cum[g]; }
    const ScanPlan plan = scan_plan(n, sm_count());
    if (plan.tpc > (uint32_t)MAX_TPC_SMEM) return HMC_ERR_SIZE;   // cannot happen: scan_plan caps it
    double4* slice_tot = reinterpret_cast<double4*>(ws.scan_status);
    double4* chunk_tot = slice_tot + plan.nslices;
    potential_reduce_kernel<<<plan.nchunks, SCAN_THREADS, 0, st>>>(r, m, n, plan, slice_tot, chunk_tot);
    HMC_LAUNCH_CHECK();
    potential_apply_kernel<<<plan.nchunks, SCAN_THREADS, 0, st>>>(r, m, phi, m_cum, n, G, plan, slice_tot, chunk_tot,
                                                                  reinterpret_cast<const double4*>(ext_tot), nranks, rank, push);
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

}  // namespace hmc

// ---- hmc_potential_static: S2 with its scratch inside the library image (include/hmc.h) -----------------------
// For callers that may not allocate device memory (a plug-in inside a host program that owns the allocator, a
// callback under the allocator's lock, a loop that cannot afford cudaMalloc's device synchronisation): the partial
// sums the reduce launch hands to the apply launch live in this array instead of a caller's workspace.
// Layout: slice totals [STATIC_MAX_SLICES] double4, then chunk totals [STATIC_MAX_CHUNKS] double4.
// One copy per GPU that loads the library, held until the process exits.  Every call on a device shares it:
// nothing needs clearing between calls (the reduce launch writes every entry the apply launch reads), but calls
// that overlap on the GPU race on it.
static constexpr uint32_t STATIC_MAX_SLICES = (uint32_t)(HMC_STATIC_MAX_N / hmc::SLICE);   // 16384
static constexpr uint32_t STATIC_MAX_CHUNKS = 1024;                                         // CTAs of a launch: 3 per SM
static_assert((STATIC_MAX_SLICES + STATIC_MAX_CHUNKS) * sizeof(double4) == HMC_STATIC_SCRATCH_BYTES, "hmc.h states the size");
static_assert(HMC_STATIC_MAX_N % hmc::SLICE == 0 && HMC_STATIC_MAX_N <= HMC_MAX_N, "limit is a whole number of slices");

static __device__ __align__(256) unsigned char g_static_scratch[HMC_STATIC_SCRATCH_BYTES];

// In host code `g_static_scratch` names a host-side shadow of the symbol, not device memory: a kernel handed
// &g_static_scratch would fault (or scribble on host memory where the GPU can reach it).  The address the kernels
// need comes from cudaGetSymbolAddress, which answers for the CURRENT device; it is looked up once per device and kept.
static hmc_status static_scratch_address(double4** out)
{
    static std::atomic<void*> cached[64];                   // zero-initialised; one slot per device ordinal
    int dev = 0;
    HMC_CUDA_TRY(cudaGetDevice(&dev));
    const bool slot = dev >= 0 && dev < 64;
    void* p = slot ? cached[dev].load(std::memory_order_acquire) : nullptr;
    if (p == nullptr) {
        HMC_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_scratch));   // same answer from every thread: no lock needed
        if (p == nullptr) return HMC_ERR_CUDA;
        if (slot) cached[dev].store(p, std::memory_order_release);
    }
    *out = static_cast<double4*>(p);
    return HMC_OK;
}

extern "C" hmc_status hmc_potential_static(uint64_t n, double G, const double* r_sorted, const double* m_sorted,
                                           double* phi, double* m_cum, void* cuda_stream)
{
    using namespace hmc;
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    if (n > HMC_STATIC_MAX_N) return HMC_ERR_STATIC_LIMIT;
    if (n == 0) return HMC_OK;
    if (!r_sorted || !m_sorted || !phi || !m_cum) return HMC_ERR_NULL;
    if (misaligned(r_sorted, 8) || misaligned(m_sorted, 8) || misaligned(phi, 8) || misaligned(m_cum, 8)) return HMC_ERR_ALIGN;
    const ScanPlan plan = scan_plan(n, sm_count());         // what potential() below will compute again
    if (plan.nslices > STATIC_MAX_SLICES || plan.nchunks > STATIC_MAX_CHUNKS) return HMC_ERR_STATIC_LIMIT;
    double4* scratch = nullptr;
    const hmc_status s = static_scratch_address(&scratch);
    if (s != HMC_OK) return s;
    // potential() places the chunk totals right behind the plan.nslices slice totals: both fit by the check above
    Workspace ws{};
    ws.scan_status = reinterpret_cast<double*>(scratch);
    return potential(n, G, r_sorted, m_sorted, phi, m_cum, nullptr, 0, 0, ws, static_cast<cudaStream_t>(cuda_stream));
}
