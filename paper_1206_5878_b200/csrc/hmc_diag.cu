// hmc_diag.cu -- diagnostics on the radius-sorted arrays (PAPER.md:140, :346 Eq. 20, :354;
// SURVEY.md 8(f) item 4; R15-R17): total mass, kinetic and potential energy, virial
// ratio, half-mass and Lagrange radii, half-mass relaxation time.
//
// One streaming pass (32 bytes per star) accumulates T = sum m (v_r^2 + v_t^2)/2 and
// W = sum m Phi / 2 in double-double, per thread, per warp, per CTA; a single-CTA kernel adds the
// CTA partials (again double-double, so the sums are the exact sums of the binary64 terms rounded
// once, whatever the association order), finds the Lagrange radii by bisection over M_cum (one
// thread per mass fraction) and evaluates Eq. 20.
#include "hmc_common.cuh"

namespace hmc {

static constexpr int DIAG_THREADS = 256;
static constexpr int DIAG_WARPS = DIAG_THREADS / 32;

__device__ __forceinline__ dd dd_shfl_xor_(dd v, int mask)
{
    return dd{ __shfl_xor_sync(0xffffffffu, v.hi, mask), __shfl_xor_sync(0xffffffffu, v.lo, mask) };
}

// partials[cta] = (T.hi, T.lo, W.hi, W.lo)
__global__ void __launch_bounds__(DIAG_THREADS)
diag_reduce_kernel(const double* __restrict__ v_r, const double* __restrict__ v_t, const double* __restrict__ m,
                   const double* __restrict__ phi, uint64_t n, double4* __restrict__ partials)
{
    __shared__ dd sT[DIAG_WARPS], sW[DIAG_WARPS];
    dd aT{ 0.0, 0.0 }, aW{ 0.0, 0.0 };
    const uint64_t stride = (uint64_t)gridDim.x * DIAG_THREADS;
    for (uint64_t a = (uint64_t)blockIdx.x * DIAG_THREADS + threadIdx.x; a < n; a += stride) {
        const double vr = __ldcs(v_r + a), vt = __ldcs(v_t + a), mm = __ldcs(m + a), ph = __ldcs(phi + a);
        aT = dd_add_d(aT, mm * (0.5 * (vr * vr + vt * vt)));      // the oracle's term expressions (R15)
        aW = dd_add_d(aW, 0.5 * (mm * ph));
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { aT = dd_add(aT, dd_shfl_xor_(aT, d)); aW = dd_add(aW, dd_shfl_xor_(aW, d)); }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) { sT[warp] = aT; sW[warp] = aW; }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < DIAG_WARPS; ++w) { aT = dd_add(aT, sT[w]); aW = dd_add(aW, sW[w]); }
        partials[blockIdx.x] = make_double4(aT.hi, aT.lo, aW.hi, aW.lo);
    }
}

struct DiagFractions {
    double f[HMC_DIAG_MAX_FRACTIONS];
    int n;
};

// r_k of the first star k with M_k >= f M_N, the outermost star if there is none (M_cum ascending)
__device__ __forceinline__ double lagrange_radius(const double* __restrict__ r, const double* __restrict__ m_cum,
                                                  uint64_t n, double f)
{
    const double target = f * __ldg(m_cum + (n - 1));
    uint64_t lo = 0, hi = n - 1;                       // answer in [lo, hi]
    while (lo < hi) {
        const uint64_t mid = lo + (hi - lo) / 2;
        if (__ldg(m_cum + mid) >= target) hi = mid; else lo = mid + 1;
    }
    return __ldg(r + lo);
}

__global__ void __launch_bounds__(DIAG_THREADS)
diag_final_kernel(const double4* __restrict__ partials, int nparts, const double* __restrict__ r,
                  const double* __restrict__ m_cum, uint64_t n, double G, DiagFractions fr, double* __restrict__ out)
{
    __shared__ dd sT[DIAG_WARPS], sW[DIAG_WARPS];
    __shared__ double s_rh;
    dd aT{ 0.0, 0.0 }, aW{ 0.0, 0.0 };
    for (int i = threadIdx.x; i < nparts; i += DIAG_THREADS) {
        const double4 p = partials[i];
        aT = dd_add(aT, dd{ p.x, p.y });
        aW = dd_add(aW, dd{ p.z, p.w });
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { aT = dd_add(aT, dd_shfl_xor_(aT, d)); aW = dd_add(aW, dd_shfl_xor_(aW, d)); }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) { sT[warp] = aT; sW[warp] = aW; }
    // one thread per requested mass fraction; thread fr.n takes the half-mass radius
    if ((int)threadIdx.x < fr.n) out[HMC_DIAG_LAGRANGE + threadIdx.x] = lagrange_radius(r, m_cum, n, fr.f[threadIdx.x]);
    if ((int)threadIdx.x == fr.n) s_rh = lagrange_radius(r, m_cum, n, 0.5);
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < DIAG_WARPS; ++w) { aT = dd_add(aT, sT[w]); aW = dd_add(aW, sW[w]); }
        const double M = __ldg(m_cum + (n - 1)), T = aT.hi, W = aW.hi, rh = s_rh;
        out[HMC_DIAG_M] = M;
        out[HMC_DIAG_T] = T;
        out[HMC_DIAG_W] = W;
        out[HMC_DIAG_ETOT] = T + W;
        out[HMC_DIAG_VIRIAL] = (2.0 * T) / fabs(W);
        out[HMC_DIAG_RH] = rh;
        out[HMC_DIAG_TRH] = ((0.138 * (double)n) / log(0.1 * (double)n)) * sqrt(((rh * rh) * rh) / (G * M));   // Eq. 20
    }
}

hmc_status diagnostics(uint64_t n, double G, const double* r, const double* v_r, const double* v_t, const double* m,
                       const double* phi, const double* m_cum, int nfrac, const double* fractions, double* out,
                       const Workspace& ws, cudaStream_t st)
{
    const int sms = sm_count();
    const uint64_t scan_tiles = (n + SCAN_TILE - 1) / SCAN_TILE;           // the partials live in the scan scratch
    int blocks = (int)umin64((n + DIAG_THREADS - 1) / DIAG_THREADS, (uint64_t)sms * 8);
    blocks = (int)umin64((uint64_t)blocks, scan_tiles * 4);                // 2 * tiles * 64 B available, 32 B used per CTA
    if (blocks < 1) blocks = 1;
    double4* partials = reinterpret_cast<double4*>(ws.scan_status);
    diag_reduce_kernel<<<blocks, DIAG_THREADS, 0, st>>>(v_r, v_t, m, phi, n, partials);
    HMC_LAUNCH_CHECK();
    DiagFractions fr{};
    fr.n = nfrac;
    for (int i = 0; i < nfrac; ++i) fr.f[i] = fractions[i];
    diag_final_kernel<<<1, DIAG_THREADS, 0, st>>>(partials, blocks, r, m_cum, n, G, fr, out);
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

}  // namespace hmc
