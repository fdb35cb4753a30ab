// hmc_orbit.cu -- S3 turning points and S4 new-radius draw (Appendix A).
//
// The paper's GPU port ran one thread per star with plain bisection over the (r, Phi) arrays in
// global memory.  What is kept: one thread per star, SoA streams, coalesced
// per-star loads and stores.  What differs:
//  * The bracket predicate "Q(r_j) < 0" is monotone on either side of the star (Q is concave in
//    1/r), so ANY search order finds the same bracket.  The search therefore descends a GLOBAL
//    implicit binary tree over node numbers (the pivot of an open interval is its element with
//    the most trailing zero bits) instead of bisecting [0,k] / [k,N+1] per star: all stars share
//    the upper levels of that tree.  Nodes whose number is a multiple of 2^t are staged once per
//    CTA in shared memory (up to 216 KB); the remaining t levels come from an interleaved
//    (r_j, Phi_j) table, one 16-byte load per probe.
//  * Random numbers are Philox4x32-10 keyed by (seed, step, star id), not per-thread streams.
#include "hmc_common.cuh"

namespace hmc {

static constexpr int ORB_THREADS = 1024;
static constexpr uint32_t COARSE_CAP_RPHI = 13824;   // (r, Phi) pairs: 216 KB
static constexpr uint32_t COARSE_CAP_R = 27648;      // r only:        216 KB

static int coarse_shift(uint64_t n, uint32_t cap)
{
    int t = 0;
    while ((n >> t) + 1 > cap) ++t;
    return t;
}

// element of the open interval (lo, hi), hi - lo > 1, with the most trailing zeros
__device__ __forceinline__ uint32_t pivot(uint32_t lo, uint32_t hi)
{
    uint32_t b = hi - 1;
    uint32_t x = lo ^ b;                       // lo < b: highest differing bit is set in b
    int hb = 31 - __clz(x);
    return b & (0xffffffffu << hb);
}

__global__ void __launch_bounds__(256) build_rphi_kernel(const double* __restrict__ r, const double* __restrict__ phi,
                                                         double2* __restrict__ rphi, uint64_t n)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        rphi[i] = make_double2(r[i], phi[i]);
}

// ---- S3 ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(ORB_THREADS, 1)
turning_points_kernel(uint32_t n, double G, const double* __restrict__ r, const double* __restrict__ v_r,
                      const double* __restrict__ v_t, const double* __restrict__ phi,
                      const double* __restrict__ m_cum, const double2* __restrict__ rphi, int shift,
                      double* __restrict__ E_out, double* __restrict__ J_out, double* __restrict__ rmin_out,
                      double* __restrict__ rmax_out, uint32_t* __restrict__ kmin_out, uint32_t* __restrict__ kmax_out,
                      uint8_t* __restrict__ status_out, unsigned long long* __restrict__ counters)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* coarse = reinterpret_cast<double2*>(smem_raw);     // coarse[c] = node c << shift, c >= 1
    const uint32_t ncoarse = n >> shift;
    for (uint32_t c = threadIdx.x + 1; c <= ncoarse; c += ORB_THREADS) coarse[c] = rphi[((uint64_t)c << shift) - 1];
    __syncthreads();
    const uint32_t low_mask = (1u << shift) - 1u;

    const uint32_t stride = gridDim.x * ORB_THREADS;
    for (uint32_t a = blockIdx.x * ORB_THREADS + threadIdx.x; a < n; a += stride) {
        const uint32_t k = a + 1;
        const double rk = r[a], vr = v_r[a], vt = v_t[a], phik = phi[a];
        const double E = phik + 0.5 * (vr * vr + vt * vt);      // Eq. 16
        const double J = rk * vt;
        const double J2 = J * J;
        unsigned st = 0;
        if (!(E < 0.0)) st |= HMC_STAR_UNBOUND;
        if (J2 == 0.0) st |= HMC_STAR_RADIAL;
        double rmin, rmax;
        uint32_t kmin, kmax;
        if (st) {
            rmin = (st & HMC_STAR_RADIAL) ? 0.0 : rk;
            rmax = (st & HMC_STAR_UNBOUND) ? __longlong_as_double(0x7ff0000000000000ll) : rk;
            kmin = k - 1; kmax = k;
        } else {
            // pericentre bracket: Q_lo < 0 <= Q_hi
            uint32_t lo = 0, hi = k;
            while (hi - lo > 1) {
                uint32_t p = pivot(lo, hi);
                double2 e = (p & low_mask) ? __ldg(rphi + (p - 1)) : coarse[p >> shift];
                bool neg = 2.0 * ((E - e.y) * (e.x * e.x)) < J2;      // Q(r_p) < 0, division-free (R2)
                if (neg) lo = p; else hi = p;
            }
            kmin = lo;
            // apocentre bracket: Q_lo >= 0 > Q_hi
            lo = k; hi = n + 1;
            while (hi - lo > 1) {
                uint32_t p = pivot(lo, hi);
                double2 e = (p & low_mask) ? __ldg(rphi + (p - 1)) : coarse[p >> shift];
                bool neg = 2.0 * ((E - e.y) * (e.x * e.x)) < J2;
                if (neg) hi = p; else lo = p;
            }
            kmax = lo;
            // closed-form roots of Q(u) = 2C + 2Bu - J^2 u^2 in the bracketing shells (R3)
            double B, C;
            if (kmin == 0) { B = 0.0; C = E - phi[0]; }
            else {
                double2 e = __ldg(rphi + (kmin - 1));
                B = G * __ldg(m_cum + (kmin - 1));
                C = (E - e.y) - B * (1.0 / e.x);
            }
            double D = B * B + 2.0 * (J2 * C);
            if (D < 0.0) D = 0.0;
            rmin = J2 / (B + sqrt(D));
            {
                double2 e = __ldg(rphi + (kmax - 1));               // kmax >= k >= 1
                B = G * __ldg(m_cum + (kmax - 1));
                C = (E - e.y) - B * (1.0 / e.x);
            }
            D = B * B + 2.0 * (J2 * C);
            if (D < 0.0) D = 0.0;
            if (C < 0.0) rmax = (B + sqrt(D)) / (-2.0 * C);
            else { rmax = __longlong_as_double(0x7ff0000000000000ll); st |= HMC_STAR_DEGENERATE; }
        }
        E_out[a] = E; J_out[a] = J; rmin_out[a] = rmin; rmax_out[a] = rmax;
        kmin_out[a] = kmin; kmax_out[a] = kmax; status_out[a] = (uint8_t)st;
        if (st && counters) {
            if (st & HMC_STAR_UNBOUND) atomicAdd(counters + HMC_CNT_UNBOUND, 1ull);
            if (st & HMC_STAR_RADIAL) atomicAdd(counters + HMC_CNT_RADIAL, 1ull);
            if (st & HMC_STAR_DEGENERATE) atomicAdd(counters + HMC_CNT_DEGENERATE, 1ull);
        }
    }
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

// ---- S4 ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(ORB_THREADS, 1)
sample_new_radius_kernel(uint32_t n, double G, uint32_t seed_lo, uint32_t seed_hi, uint32_t step,
                         const double* __restrict__ r, const double* __restrict__ phi,
                         const double* __restrict__ m_cum, int shift, const double* __restrict__ v_r,
                         const double* __restrict__ v_t, const double* __restrict__ E_in,
                         const double* __restrict__ J_in, const double* __restrict__ rmin_in,
                         const double* __restrict__ rmax_in, const uint32_t* __restrict__ kmin_in,
                         const uint32_t* __restrict__ kmax_in, const uint32_t* __restrict__ id,
                         const uint8_t* __restrict__ status_in, double* __restrict__ r_new,
                         double* __restrict__ v_r_new, double* __restrict__ v_t_new, uint16_t* __restrict__ n_try,
                         uint8_t* __restrict__ status_out, unsigned long long* __restrict__ counters)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* coarse = reinterpret_cast<double*>(smem_raw);       // coarse[c] = r of node c << shift
    const uint32_t ncoarse = n >> shift;
    for (uint32_t c = threadIdx.x + 1; c <= ncoarse; c += ORB_THREADS) coarse[c] = r[((uint64_t)c << shift) - 1];
    __syncthreads();
    const uint32_t low_mask = (1u << shift) - 1u;
    const double two_m53 = 1.0 / 9007199254740992.0;
    unsigned long long my_trials = 0;

    const uint32_t stride = gridDim.x * ORB_THREADS;
    for (uint32_t a = blockIdx.x * ORB_THREADS + threadIdx.x; a < n; a += stride) {
        unsigned st = status_in[a];
        double out_r = r[a], out_vr = v_r[a], out_vt = v_t[a];
        uint32_t used = 0;
        if (!(st & (HMC_STAR_UNBOUND | HMC_STAR_RADIAL | HMC_STAR_DEGENERATE))) {
            const double E = E_in[a], J = J_in[a], J2 = J * J;
            const double rmin = rmin_in[a], rmax = rmax_in[a];
            const uint32_t kmin = kmin_in[a], kmax = kmax_in[a];
            const double delta = rmax - rmin;
            bool ok = delta > 0.0;
            double F = 0.0;
            if (ok) {
                double Bmin = (kmin == 0) ? 0.0 : G * __ldg(m_cum + (kmin - 1));
                double Bmax = (kmax == 0) ? 0.0 : G * __ldg(m_cum + (kmax - 1));
                double q1 = (2.0 * (J2 / rmin - Bmin)) / (rmin * rmin);      // Q'(r_min) in shell k_min
                double q2 = (2.0 * (J2 / rmax - Bmax)) / (rmax * rmax);      // Q'(r_max) in shell k_max
                ok = (q1 > 0.0) && (q2 < 0.0);
                if (ok) F = 1.2 * fmax(sqrt((3.0 * delta) / q1), sqrt((3.0 * delta) / (-q2)));
            }
            if (!ok) st |= HMC_STAR_CIRCULAR;
            else {
                const double mid = 0.5 * (rmin + rmax);
                const double quarter = 0.25 * delta, three_q = 0.75 * delta;
                const uint32_t sid = id[a];
                bool accepted = false, have_good = false;
                double good_r = 0.0, good_Q = 0.0;
                uint32_t good_w3 = 0, t = 0;
                for (; t < HMC_T_MAX; ++t) {
                    uint32_t w[4];
                    philox4x32_10(sid, 0u, step, t, seed_lo, seed_hi, w);
                    double X = (double)((((unsigned long long)w[0] << 32) | w[1]) >> 11) * two_m53;
                    double Xp = (double)((((unsigned long long)w[2] << 32) | w[3]) >> 11) * two_m53;
                    double s = 2.0 * X - 1.0;
                    double r0 = mid + quarter * (3.0 * s - (s * s) * s);
                    // shell of r0: j = #{ i : r_i <= r0 } clamped to [kmin, kmax]
                    uint32_t lo = kmin, hi = kmax + 1;
                    while (hi - lo > 1) {
                        uint32_t p = pivot(lo, hi);
                        double rp = (p & low_mask) ? __ldg(r + (p - 1)) : coarse[p >> shift];
                        if (rp <= r0) lo = p; else hi = p;
                    }
                    double phi0;
                    if (lo == 0) phi0 = __ldg(phi);
                    else phi0 = __ldg(phi + (lo - 1)) - (G * __ldg(m_cum + (lo - 1))) * (1.0 / r0 - 1.0 / __ldg(r + (lo - 1)));
                    double Q0 = 2.0 * (E - phi0) - J2 / (r0 * r0);
                    if (Q0 > 0.0) {
                        double g = (three_q * (1.0 - s * s)) / sqrt(Q0);
                        have_good = true; good_r = r0; good_Q = Q0; good_w3 = w[3];
                        if (g > F) st |= HMC_STAR_CLIPPED;
                        if (F * Xp < g) { accepted = true; break; }
                    }
                }
                used = accepted ? t + 1 : HMC_T_MAX;
                my_trials += used;
                if (!accepted) st |= HMC_STAR_MAXTRIES;
                if (have_good) {
                    out_r = good_r;
                    out_vt = J / good_r;
                    double vrn = sqrt(good_Q);
                    out_vr = (good_w3 & 1u) ? -vrn : vrn;
                }
            }
        }
        r_new[a] = out_r; v_r_new[a] = out_vr; v_t_new[a] = out_vt;
        if (n_try) n_try[a] = (uint16_t)used;
        status_out[a] = (uint8_t)st;
        if (counters && (st & (HMC_STAR_CIRCULAR | HMC_STAR_MAXTRIES | HMC_STAR_CLIPPED))) {
            if (st & HMC_STAR_CIRCULAR) atomicAdd(counters + HMC_CNT_CIRCULAR, 1ull);
            if (st & HMC_STAR_MAXTRIES) atomicAdd(counters + HMC_CNT_MAXTRIES, 1ull);
            if (st & HMC_STAR_CLIPPED) atomicAdd(counters + HMC_CNT_CLIPPED, 1ull);
        }
    }
    if (counters) {
        // one atomic per warp for the trial count
        for (int off = 16; off > 0; off >>= 1) my_trials += __shfl_down_sync(0xffffffffu, my_trials, off);
        if ((threadIdx.x & 31) == 0 && my_trials) atomicAdd(counters + HMC_CNT_TRIALS, my_trials);
    }
}

// ---- host side --------------------------------------------------------------------------------
hmc_status turning_points(uint64_t n, double G, const double* r, const double* v_r, const double* v_t,
                          const double* phi, const double* m_cum, double* E, double* J, double* r_min,
                          double* r_max, uint32_t* k_min, uint32_t* k_max, uint8_t* status, uint64_t* counters,
                          const Workspace& ws, cudaStream_t st)
{
    const int sms = sm_count();
    const int shift = coarse_shift(n, COARSE_CAP_RPHI);
    const size_t smem = ((n >> shift) + 1) * sizeof(double2);
    static bool attr_done = false;
    if (!attr_done) {
        HMC_CUDA_TRY(cudaFuncSetAttribute(turning_points_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)(COARSE_CAP_RPHI * sizeof(double2))));
        attr_done = true;
    }
    int blocks = (int)umin64((n + 255) / 256, (uint64_t)sms * 8);
    build_rphi_kernel<<<blocks, 256, 0, st>>>(r, phi, ws.rphi, n);
    HMC_LAUNCH_CHECK();
    blocks = (int)umin64((n + ORB_THREADS - 1) / ORB_THREADS, (uint64_t)sms);
    turning_points_kernel<<<blocks, ORB_THREADS, smem, st>>>((uint32_t)n, G, r, v_r, v_t, phi, m_cum, ws.rphi, shift, E,
                                                            J, r_min, r_max, k_min, k_max, status,
                                                            reinterpret_cast<unsigned long long*>(counters));
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

hmc_status sample_new_radius(uint64_t n, double G, uint64_t seed, uint32_t step, const double* r,
                             const double* phi, const double* m_cum, const double* v_r, const double* v_t,
                             const double* E, const double* J, const double* r_min, const double* r_max,
                             const uint32_t* k_min, const uint32_t* k_max, const uint32_t* id,
                             const uint8_t* status_in, double* r_new, double* v_r_new, double* v_t_new,
                             uint16_t* n_try, uint8_t* status_out, uint64_t* counters, const Workspace& ws,
                             cudaStream_t st)
{
    (void)ws;
    const int sms = sm_count();
    const int shift = coarse_shift(n, COARSE_CAP_R);
    const size_t smem = ((n >> shift) + 1) * sizeof(double);
    static bool attr_done = false;
    if (!attr_done) {
        HMC_CUDA_TRY(cudaFuncSetAttribute(sample_new_radius_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)(COARSE_CAP_R * sizeof(double))));
        attr_done = true;
    }
    int blocks = (int)umin64((n + ORB_THREADS - 1) / ORB_THREADS, (uint64_t)sms);
    sample_new_radius_kernel<<<blocks, ORB_THREADS, smem, st>>>(
        (uint32_t)n, G, (uint32_t)seed, (uint32_t)(seed >> 32), step, r, phi, m_cum, shift, v_r, v_t, E, J, r_min, r_max,
        k_min, k_max, id, status_in, r_new, v_r_new, v_t_new, n_try, status_out,
        reinterpret_cast<unsigned long long*>(counters));
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

}  // namespace hmc
