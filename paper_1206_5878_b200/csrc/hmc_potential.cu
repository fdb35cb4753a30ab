// hmc_potential.cu -- S2: Phi_k = -G (M_k / r_k + S_k) on the radius-sorted arrays.
//
// The paper computes Phi by the backward recursion Eq. 2-5 and calls it "inherently sequential"
// (PAPER.md:185).  Here it is two single-pass prefix scans with decoupled look-back:
//   pass A (tiles taken from the outside in):  S_k = sum_{i>k} fl(m_i / r_i)   -> written to phi[]
//   pass B (tiles taken from the inside out):  M_k = sum_{i<=k} m_i, then
//                                              Phi_k = -(G * (M_k / r_k + S_k)) overwrites phi[k].
// Both running sums are double-double (106 bits) and rounded once, so the result does not depend
// on the association order of the scan (R1p).
#include "hmc_common.cuh"

namespace hmc {

static constexpr int SCAN_THREADS = 256;
static constexpr int SCAN_ITEMS = SCAN_TILE / SCAN_THREADS;   // 8
static constexpr int SCAN_WARPS = SCAN_THREADS / 32;

// tile status record: 8 doubles = 64 bytes; word 0 carries the flag (as a double: 0, 1, 2)
//   [0] flag  [1] agg.hi [2] agg.lo [3] inc.hi [4] inc.lo
static constexpr double SCAN_EMPTY = 0.0, SCAN_AGG = 1.0, SCAN_INC = 2.0;

// REVERSE = true : logical position p <-> array index n-1-p, value fl(m/r), output the EXCLUSIVE sum
// REVERSE = false: logical position p <-> array index p,     value m,      output the INCLUSIVE sum
template <bool REVERSE>
__global__ void __launch_bounds__(SCAN_THREADS)
potential_scan_kernel(const double* __restrict__ r, const double* __restrict__ m, double* __restrict__ phi,
                      double* __restrict__ m_cum, uint64_t n, double G, double* __restrict__ status,
                      uint32_t* __restrict__ ticket)
{
    __shared__ dd warp_tot[SCAN_WARPS];
    __shared__ dd tile_prefix;
    __shared__ uint32_t s_tile;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint64_t tile = s_tile;
    const uint64_t p0 = tile * SCAN_TILE + (uint64_t)tid * SCAN_ITEMS;

    double x[SCAN_ITEMS], rr[SCAN_ITEMS];
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) {
        uint64_t p = p0 + i;
        if (p < n) {
            uint64_t a = REVERSE ? (n - 1 - p) : p;
            double mm = m[a];
            rr[i] = r[a];
            x[i] = REVERSE ? (mm / rr[i]) : mm;
        } else {
            x[i] = 0.0; rr[i] = 1.0;
        }
    }
    // thread total
    dd tot{ 0.0, 0.0 };
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) tot = dd_add_d(tot, x[i]);
    // inclusive scan of thread totals inside the warp
    dd inc = tot;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        dd up = dd_shfl_up(inc, d);
        if (lane >= d) inc = dd_add(up, inc);
    }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    // exclusive prefix of this thread inside the tile
    dd excl{ 0.0, 0.0 };
    for (int w = 0; w < warp; ++w) excl = dd_add(excl, warp_tot[w]);
    {
        dd prev = dd_shfl_up(inc, 1);
        if (lane > 0) excl = dd_add(excl, prev);
    }
    // tile aggregate -> look-back (one thread; predecessors are always resident or finished)
    if (tid == SCAN_THREADS - 1) {
        dd agg = dd_add(excl, tot);
        double* my = status + tile * 8;
        dd pre{ 0.0, 0.0 };
        if (tile == 0) {
            st_volatile_f64(my + 3, agg.hi); st_volatile_f64(my + 4, agg.lo);
            __threadfence();
            st_volatile_f64(my, SCAN_INC);
        } else {
            st_volatile_f64(my + 1, agg.hi); st_volatile_f64(my + 2, agg.lo);
            __threadfence();
            st_volatile_f64(my, SCAN_AGG);
            for (int64_t t = (int64_t)tile - 1; t >= 0; --t) {
                const double* q = status + (uint64_t)t * 8;
                double f;
                do { f = ld_volatile_f64(q); } while (f == SCAN_EMPTY);
                __threadfence();
                if (f == SCAN_INC) {
                    pre = dd_add(pre, dd{ ld_volatile_f64(q + 3), ld_volatile_f64(q + 4) });
                    break;
                }
                pre = dd_add(pre, dd{ ld_volatile_f64(q + 1), ld_volatile_f64(q + 2) });
            }
            dd incl = dd_add(pre, agg);
            st_volatile_f64(my + 3, incl.hi); st_volatile_f64(my + 4, incl.lo);
            __threadfence();
            st_volatile_f64(my, SCAN_INC);
        }
        tile_prefix = pre;
    }
    __syncthreads();
    dd run = dd_add(tile_prefix, excl);
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) {
        uint64_t p = p0 + i;
        if (REVERSE) {
            if (p < n) phi[n - 1 - p] = run.hi;          // S_k: exclusive suffix sum, rounded once
            run = dd_add_d(run, x[i]);
        } else {
            run = dd_add_d(run, x[i]);
            if (p < n) {
                double M = run.hi;                        // M_k: inclusive prefix sum, rounded once
                double S = phi[p];
                m_cum[p] = M;
                phi[p] = -(G * (M / rr[i] + S));          // Eq. 1 at r = r_k
            }
        }
    }
}

hmc_status potential(uint64_t n, double G, const double* r, const double* m, double* phi, double* m_cum,
                     const Workspace& ws, cudaStream_t st)
{
    const uint64_t tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    HMC_CUDA_TRY(cudaMemsetAsync(ws.scan_status, 0, 2 * tiles * 8 * 8, st));
    HMC_CUDA_TRY(cudaMemsetAsync(ws.tickets + 16, 0, 2 * 4, st));
    potential_scan_kernel<true><<<(unsigned)tiles, SCAN_THREADS, 0, st>>>(r, m, phi, m_cum, n, G, ws.scan_status,
                                                                         ws.tickets + 16);
    HMC_LAUNCH_CHECK();
    potential_scan_kernel<false><<<(unsigned)tiles, SCAN_THREADS, 0, st>>>(r, m, phi, m_cum, n, G,
                                                                          ws.scan_status + tiles * 8, ws.tickets + 17);
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

}  // namespace hmc
