// hmc_potential.cu -- S2: Phi_k = -G (M_k / r_k + S_k) on the radius-sorted arrays.
//
// The paper computes Phi by the backward recursion Eq. 2-5 and calls it "inherently sequential"
// (PAPER.md:185).  Here it is a reduce-then-scan over tiles of 2048 stars, three launches:
//   1. potential_reduce_kernel : per tile, T_m = sum m_i and T_t = sum fl(m_i / r_i)
//   2. potential_totals_kernel : one CTA; exclusive prefix of T_m (inside out) and exclusive
//                                suffix of T_t (outside in) over the tiles
//   3. potential_apply_kernel  : per tile, forward scan of m and backward scan of m/r in
//                                registers, M_k and S_k rounded once, Phi_k = -(G*(M_k/r_k + S_k)).
// Every partial sum is double-double (106 bits), so M_k and S_k are the exact sums rounded once
// and do not depend on the association order (R1p).  There is no inter-CTA waiting.
// Launch 3 walks the tiles in the opposite order to launch 1, so the part of r, m that is still
// in the 126 MB L2 is read from there.
#include "hmc_common.cuh"

namespace hmc {

static constexpr int SCAN_THREADS = 128;
static constexpr int SCAN_ITEMS = SCAN_TILE / SCAN_THREADS;   // 16
static constexpr int SCAN_WARPS = SCAN_THREADS / 32;
static constexpr int TOT_THREADS = 1024;

__device__ __forceinline__ dd dd_shfl_xor(dd v, int mask)
{
    return dd{ __shfl_xor_sync(0xffffffffu, v.hi, mask), __shfl_xor_sync(0xffffffffu, v.lo, mask) };
}
__device__ __forceinline__ dd dd_shfl_down(dd v, int delta)
{
    return dd{ __shfl_down_sync(0xffffffffu, v.hi, delta), __shfl_down_sync(0xffffffffu, v.lo, delta) };
}

// ---- 1. tile totals ---------------------------------------------------------------------------
// totals[tile] = (T_m.hi, T_m.lo, T_t.hi, T_t.lo).  Element order inside a tile is irrelevant for
// a sum, so the loads are fully coalesced 16-byte loads.
__global__ void __launch_bounds__(SCAN_THREADS)
potential_reduce_kernel(const double* __restrict__ r, const double* __restrict__ m, uint64_t n,
                        double4* __restrict__ totals)
{
    __shared__ dd sm_m[SCAN_WARPS], sm_t[SCAN_WARPS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint64_t base = (uint64_t)blockIdx.x * SCAN_TILE;
    dd am{ 0.0, 0.0 }, at{ 0.0, 0.0 };
    if (base + SCAN_TILE <= n && ((reinterpret_cast<uintptr_t>(r) | reinterpret_cast<uintptr_t>(m)) & 15) == 0) {
        const double2* r2 = reinterpret_cast<const double2*>(r + base);
        const double2* m2 = reinterpret_cast<const double2*>(m + base);
        double2 rv[SCAN_ITEMS / 2], mv[SCAN_ITEMS / 2];
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS / 2; ++i) { rv[i] = __ldg(r2 + i * SCAN_THREADS + tid); mv[i] = __ldg(m2 + i * SCAN_THREADS + tid); }
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS / 2; ++i) {
            am = dd_add_d(am, mv[i].x); am = dd_add_d(am, mv[i].y);
            at = dd_add_d(at, mv[i].x / rv[i].x); at = dd_add_d(at, mv[i].y / rv[i].y);
        }
    } else {
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS; ++i) {
            uint64_t a = base + (uint64_t)i * SCAN_THREADS + tid;
            if (a < n) { double mm = m[a]; am = dd_add_d(am, mm); at = dd_add_d(at, mm / r[a]); }
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { am = dd_add(am, dd_shfl_xor(am, d)); at = dd_add(at, dd_shfl_xor(at, d)); }
    if (lane == 0) { sm_m[warp] = am; sm_t[warp] = at; }
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int w = 1; w < SCAN_WARPS; ++w) { am = dd_add(am, sm_m[w]); at = dd_add(at, sm_t[w]); }
        totals[blockIdx.x] = make_double4(am.hi, am.lo, at.hi, at.lo);
    }
}

// ---- 2. scan of the tile totals (single CTA) ---------------------------------------------------
// in : totals[tile] = (T_m, T_t);  out: totals[tile] = (prefix of T_m over tiles < tile,
//                                                       suffix of T_t over tiles > tile)
__global__ void __launch_bounds__(TOT_THREADS)
potential_totals_kernel(double4* __restrict__ totals, uint32_t ntiles)
{
    __shared__ dd sm_m[TOT_THREADS / 32], sm_t[TOT_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t per = (ntiles + TOT_THREADS - 1) / TOT_THREADS;
    const uint32_t lo = min(ntiles, (uint32_t)tid * per), hi = min(ntiles, lo + per);
    dd tm{ 0.0, 0.0 }, tt{ 0.0, 0.0 };
    for (uint32_t i = lo; i < hi; ++i) {
        double4 v = totals[i];
        tm = dd_add(tm, dd{ v.x, v.y });
        tt = dd_add(tt, dd{ v.z, v.w });
    }
    // inclusive scans over threads: forward for m, backward for t
    dd im = tm, it = tt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        dd up = dd_shfl_up(im, d);
        if (lane >= d) im = dd_add(up, im);
        dd dn = dd_shfl_down(it, d);
        if (lane + d < 32) it = dd_add(it, dn);
    }
    if (lane == 31) sm_m[warp] = im;
    if (lane == 0) sm_t[warp] = it;
    __syncthreads();
    dd em{ 0.0, 0.0 }, et{ 0.0, 0.0 };
    for (int w = 0; w < warp; ++w) em = dd_add(em, sm_m[w]);
    for (int w = TOT_THREADS / 32 - 1; w > warp; --w) et = dd_add(et, sm_t[w]);
    {
        dd pm = dd_shfl_up(im, 1), pt = dd_shfl_down(it, 1);
        if (lane > 0) em = dd_add(em, pm);
        if (lane < 31) et = dd_add(et, pt);
    }
    // em = sum of T_m over all tiles owned by lower threads; et = sum of T_t over higher threads.
    // suffix inside the thread's own range needs the later tiles first: walk it backwards.
    dd run_t = et;
    for (uint32_t i = hi; i-- > lo;) {
        double4 v = totals[i];
        totals[i].z = run_t.hi; totals[i].w = run_t.lo;
        run_t = dd_add(run_t, dd{ v.z, v.w });
    }
    dd run_m = em;
    for (uint32_t i = lo; i < hi; ++i) {
        double4 v = totals[i];
        totals[i].x = run_m.hi; totals[i].y = run_m.lo;
        run_m = dd_add(run_m, dd{ v.x, v.y });
    }
}

// ---- 3. per-tile scans and Phi -----------------------------------------------------------------
__global__ void __launch_bounds__(SCAN_THREADS)
potential_apply_kernel(const double* __restrict__ r, const double* __restrict__ m, double* __restrict__ phi,
                       double* __restrict__ m_cum, uint64_t n, double G, const double4* __restrict__ totals,
                       uint32_t ntiles)
{
    __shared__ dd sm_m[SCAN_WARPS], sm_t[SCAN_WARPS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tile = ntiles - 1 - blockIdx.x;           // opposite order to the reduce launch
    const uint64_t p0 = (uint64_t)tile * SCAN_TILE + (uint64_t)tid * SCAN_ITEMS;
    double rr[SCAN_ITEMS], mm[SCAN_ITEMS], tt[SCAN_ITEMS];
    const bool full = (uint64_t)tile * SCAN_TILE + SCAN_TILE <= n;
    const bool al = ((reinterpret_cast<uintptr_t>(r) | reinterpret_cast<uintptr_t>(m)) & 15) == 0;
    if (full && al) {
        const double2* r2 = reinterpret_cast<const double2*>(r + p0);
        const double2* m2 = reinterpret_cast<const double2*>(m + p0);
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS / 2; ++i) {
            double2 a = __ldg(r2 + i), b = __ldg(m2 + i);
            rr[2 * i] = a.x; rr[2 * i + 1] = a.y; mm[2 * i] = b.x; mm[2 * i + 1] = b.y;
        }
    } else {
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS; ++i) {
            uint64_t p = p0 + i;
            rr[i] = (p < n) ? r[p] : 1.0;
            mm[i] = (p < n) ? m[p] : 0.0;
        }
    }
    dd tm{ 0.0, 0.0 }, ts{ 0.0, 0.0 };
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) {
        tt[i] = mm[i] / rr[i];
        tm = dd_add_d(tm, mm[i]);
        ts = dd_add_d(ts, tt[i]);
    }
    dd im = tm, it = ts;                                       // inclusive over threads: forward m, backward t
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        dd up = dd_shfl_up(im, d);
        if (lane >= d) im = dd_add(up, im);
        dd dn = dd_shfl_down(it, d);
        if (lane + d < 32) it = dd_add(it, dn);
    }
    if (lane == 31) sm_m[warp] = im;
    if (lane == 0) sm_t[warp] = it;
    __syncthreads();
    const double4 tp = totals[tile];
    dd em{ tp.x, tp.y }, et{ tp.z, tp.w };                     // everything before / after this tile
    for (int w = 0; w < warp; ++w) em = dd_add(em, sm_m[w]);
    for (int w = SCAN_WARPS - 1; w > warp; --w) et = dd_add(et, sm_t[w]);
    {
        dd pm = dd_shfl_up(im, 1), pt = dd_shfl_down(it, 1);
        if (lane > 0) em = dd_add(em, pm);
        if (lane < 31) et = dd_add(et, pt);
    }
    double Mk[SCAN_ITEMS], Sk[SCAN_ITEMS];
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { em = dd_add_d(em, mm[i]); Mk[i] = em.hi; }     // inclusive prefix, rounded once
#pragma unroll
    for (int i = SCAN_ITEMS - 1; i >= 0; --i) { Sk[i] = et.hi; et = dd_add_d(et, tt[i]); }  // exclusive suffix, rounded once
    double ph[SCAN_ITEMS];
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) ph[i] = -(G * (Mk[i] / rr[i] + Sk[i]));           // Eq. 1 at r = r_k
    const bool alo = ((reinterpret_cast<uintptr_t>(phi) | reinterpret_cast<uintptr_t>(m_cum)) & 15) == 0;
    if (full && alo) {
        double2* p2 = reinterpret_cast<double2*>(phi + p0);
        double2* c2 = reinterpret_cast<double2*>(m_cum + p0);
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS / 2; ++i) {
            p2[i] = make_double2(ph[2 * i], ph[2 * i + 1]);
            c2[i] = make_double2(Mk[2 * i], Mk[2 * i + 1]);
        }
    } else {
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS; ++i) {
            uint64_t p = p0 + i;
            if (p < n) { phi[p] = ph[i]; m_cum[p] = Mk[i]; }
        }
    }
}

hmc_status potential(uint64_t n, double G, const double* r, const double* m, double* phi, double* m_cum,
                     const Workspace& ws, cudaStream_t st)
{
    const uint32_t tiles = (uint32_t)((n + SCAN_TILE - 1) / SCAN_TILE);
    double4* totals = reinterpret_cast<double4*>(ws.scan_status);
    potential_reduce_kernel<<<tiles, SCAN_THREADS, 0, st>>>(r, m, n, totals);
    HMC_LAUNCH_CHECK();
    potential_totals_kernel<<<1, TOT_THREADS, 0, st>>>(totals, tiles);
    HMC_LAUNCH_CHECK();
    potential_apply_kernel<<<tiles, SCAN_THREADS, 0, st>>>(r, m, phi, m_cum, n, G, totals, tiles);
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

}  // namespace hmc
