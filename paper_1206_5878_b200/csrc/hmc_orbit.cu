// hmc_orbit.cu -- S3 turning points and S4 new-radius draw (Appendix A).
//
// The paper's GPU port ran one thread per star with plain bisection over the (r, Phi) arrays in
// global memory.  What is kept: one thread per star, SoA streams, coalesced
// per-star loads and stores.  What differs:
//
//  * Search order.  The bracket predicate "Q(r_j) < 0" is monotone on either side of the star (Q
//    is concave in 1/r), and "r_j <= r0" is monotone, so ANY search order finds the same index.
//    The searches descend a GLOBAL implicit binary tree over node numbers (the pivot of an open
//    interval is its element with the most trailing zero bits) instead of bisecting [0,k] /
//    [k,N+1] per star, so all stars share the upper levels of that tree:
//      - nodes that are multiples of 2^t  : staged once per CTA in shared memory (<= 216 KB)
//      - nodes that are multiples of 8    : a dense "mid" table (N/8 entries, L2 resident)
//      - the last three levels            : the full table; 8 consecutive entries = one line
//  * S3 runs the pericentre and the apocentre search of a star interleaved, two independent load
//    chains per thread.
//  * S4 decides most trials without touching global memory ("squeeze"): Phi is monotone in r, so
//    the shared-memory table brackets Phi(r0) and hence Q(r0) and g; a trial is rejected (or
//    provisionally accepted) when the whole bracket, widened by 1e-11, lies on one side of F X'.
//    Only provisionally accepted and undecided trials run the exact shell search and the exact
//    test, with the oracle's expressions, so the outcome is identical to evaluating every trial.
//  * Random numbers are Philox4x32-10 keyed by (seed, step, star id), not per-thread streams.
#include "hmc_common.cuh"

namespace hmc {

static constexpr int ORB_THREADS = 1024;
static constexpr uint32_t COARSE_CAP = 13824;        // (r, Phi) pairs: 216 KB
static constexpr int MID_SHIFT = 3;                  // mid tables hold every 8th node
static constexpr uint32_t MID_MASK = (1u << MID_SHIFT) - 1u;

static int coarse_shift(uint64_t n, uint32_t cap)
{
    int t = 0;
    while ((n >> t) + 2 > cap) ++t;
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

__device__ __forceinline__ double pos_inf() { return __longlong_as_double(0x7ff0000000000000ll); }

// ---- table builders ---------------------------------------------------------------------------
// rphi[a] = (r_a, Phi_a); rphi_mid[c] = node 8c = array element 8c - 1 (c >= 1)
__global__ void __launch_bounds__(256) build_rphi_kernel(const double* __restrict__ r, const double* __restrict__ phi,
                                                         double2* __restrict__ rphi, double2* __restrict__ rphi_mid,
                                                         uint64_t n)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        double2 e = make_double2(__ldcs(r + i), __ldcs(phi + i));
        rphi[i] = e;
        if (((i + 1) & MID_MASK) == 0) rphi_mid[(i + 1) >> MID_SHIFT] = e;
    }
}

// r_mid[c] = r of node 8c
__global__ void __launch_bounds__(256) build_rmid_kernel(const double* __restrict__ r, double* __restrict__ r_mid,
                                                         uint64_t n)
{
    const uint64_t nm = n >> MID_SHIFT;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t c = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x + 1; c <= nm; c += stride)
        r_mid[c] = __ldg(r + ((c << MID_SHIFT) - 1));
}

// ---- S3 ---------------------------------------------------------------------------------------
struct RPhiTable {
    const double2* full;     // [n]   node j at full[j-1]
    const double2* mid;      // [n/8+1] node 8c at mid[c]
    const double2* coarse;   // shared memory, node c << shift at coarse[c]
    uint32_t low_mask;       // (1 << shift) - 1
    int shift;
    __device__ __forceinline__ double2 global_node(uint32_t p) const
    {
        return (p & MID_MASK) ? __ldg(full + (p - 1)) : __ldg(mid + (p >> MID_SHIFT));
    }
};

// Q(r_p) < 0, division-free (R2):  2 (E - Phi_p) r_p^2 < J^2
__device__ __forceinline__ bool q_negative(double2 e, double E, double J2)
{
    return 2.0 * ((E - e.y) * (e.x * e.x)) < J2;
}

__global__ void __launch_bounds__(ORB_THREADS, 1)
turning_points_kernel(uint32_t n, double G, const double* __restrict__ r, const double* __restrict__ v_r,
                      const double* __restrict__ v_t, const double* __restrict__ phi,
                      const double* __restrict__ m_cum, const double2* __restrict__ rphi,
                      const double2* __restrict__ rphi_mid, int shift, double* __restrict__ E_out,
                      double* __restrict__ J_out, double* __restrict__ rmin_out, double* __restrict__ rmax_out,
                      uint32_t* __restrict__ kmin_out, uint32_t* __restrict__ kmax_out,
                      uint8_t* __restrict__ status_out, unsigned long long* __restrict__ counters)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* coarse = reinterpret_cast<double2*>(smem_raw);     // coarse[c] = node c << shift, c >= 1
    const uint32_t ncoarse = n >> shift;
    for (uint32_t c = threadIdx.x + 1; c <= ncoarse; c += ORB_THREADS) coarse[c] = rphi[((uint64_t)c << shift) - 1];
    __syncthreads();
    RPhiTable T{ rphi, rphi_mid, coarse, (1u << shift) - 1u, shift };

    const uint32_t stride = gridDim.x * ORB_THREADS;
    for (uint32_t a = blockIdx.x * ORB_THREADS + threadIdx.x; a < n; a += stride) {
        const uint32_t k = a + 1;
        const double rk = __ldcs(r + a), vr = __ldcs(v_r + a), vt = __ldcs(v_t + a), phik = __ldcs(phi + a);
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
            rmax = (st & HMC_STAR_UNBOUND) ? pos_inf() : rk;
            kmin = k - 1; kmax = k;
        } else {
            // pericentre bracket (lo1, hi1): Q_lo1 < 0 <= Q_hi1;  apocentre (lo2, hi2): Q_lo2 >= 0 > Q_hi2
            uint32_t lo1 = 0, hi1 = k, lo2 = k, hi2 = n + 1;
            // levels held in shared memory
            while (hi1 - lo1 > 1) {
                uint32_t p = pivot(lo1, hi1);
                if (p & T.low_mask) break;
                if (q_negative(coarse[p >> shift], E, J2)) lo1 = p; else hi1 = p;
            }
            while (hi2 - lo2 > 1) {
                uint32_t p = pivot(lo2, hi2);
                if (p & T.low_mask) break;
                if (q_negative(coarse[p >> shift], E, J2)) hi2 = p; else lo2 = p;
            }
            // remaining levels from global memory, the two searches interleaved
            while (true) {
                const bool a1 = hi1 - lo1 > 1, a2 = hi2 - lo2 > 1;
                if (!(a1 || a2)) break;
                uint32_t p1 = a1 ? pivot(lo1, hi1) : 1u, p2 = a2 ? pivot(lo2, hi2) : 1u;
                double2 e1, e2;
                if (a1) e1 = T.global_node(p1);
                if (a2) e2 = T.global_node(p2);
                if (a1) { if (q_negative(e1, E, J2)) lo1 = p1; else hi1 = p1; }
                if (a2) { if (q_negative(e2, E, J2)) hi2 = p2; else lo2 = p2; }
            }
            kmin = lo1; kmax = lo2;
            // closed-form roots of Q(u) = 2C + 2Bu - J^2 u^2 in the bracketing shells (R3)
            double2 ea = (kmin == 0) ? make_double2(1.0, __ldg(phi)) : __ldg(rphi + (kmin - 1));
            double2 eb = __ldg(rphi + (kmax - 1));                       // kmax >= k >= 1
            double Ba = (kmin == 0) ? 0.0 : G * __ldg(m_cum + (kmin - 1));
            double Bb = G * __ldg(m_cum + (kmax - 1));
            double Ca = (kmin == 0) ? (E - ea.y) : ((E - ea.y) - Ba * (1.0 / ea.x));
            double Cb = (E - eb.y) - Bb * (1.0 / eb.x);
            double D = Ba * Ba + 2.0 * (J2 * Ca);
            if (D < 0.0) D = 0.0;
            rmin = J2 / (Ba + sqrt(D));
            D = Bb * Bb + 2.0 * (J2 * Cb);
            if (D < 0.0) D = 0.0;
            if (Cb < 0.0) rmax = (Bb + sqrt(D)) / (-2.0 * Cb);
            else { rmax = pos_inf(); st |= HMC_STAR_DEGENERATE; }
        }
        __stcs(E_out + a, E); __stcs(J_out + a, J); __stcs(rmin_out + a, rmin); __stcs(rmax_out + a, rmax);
        __stcs(kmin_out + a, kmin); __stcs(kmax_out + a, kmax); status_out[a] = (uint8_t)st;
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
struct Orbit {          // per-star constants of the draw
    double E, J2, mid, quarter, three_q, F;
    uint32_t kmin, kmax, sid;
};

struct Trial {          // the random part of trial t
    double s, r0, Xp;
    uint32_t w3;
};

__device__ __forceinline__ Trial make_trial(const Orbit& o, uint32_t seed_lo, uint32_t seed_hi, uint32_t step, uint32_t t)
{
    uint32_t w[4];
    philox4x32_10(o.sid, 0u, step, t, seed_lo, seed_hi, w);
    const double two_m53 = 1.0 / 9007199254740992.0;
    double X = (double)((((unsigned long long)w[0] << 32) | w[1]) >> 11) * two_m53;
    Trial tr;
    tr.Xp = (double)((((unsigned long long)w[2] << 32) | w[3]) >> 11) * two_m53;
    tr.s = 2.0 * X - 1.0;
    tr.r0 = o.mid + o.quarter * (3.0 * tr.s - (tr.s * tr.s) * tr.s);     // replaces Eq. 14 (R7)
    tr.w3 = w[3];
    return tr;
}

struct RTable {
    const double* r;         // [n]
    const double* r_mid;     // node 8c at r_mid[c]
    const double* phi;
    const double* m_cum;
    double G;
    __device__ __forceinline__ double node_r(uint32_t p) const
    {
        return (p & MID_MASK) ? __ldg(r + (p - 1)) : __ldg(r_mid + (p >> MID_SHIFT));
    }
};

// exact evaluation of a trial, the oracle's expressions: shell j of r0 inside (lo, hi) (which must
// satisfy r_lo <= r0 < r_hi in the clamped sense), Phi(r0) by Eq. 6 anchored at j, Q0, g.
__device__ __forceinline__ void exact_trial(const RTable& T, const Orbit& o, const Trial& tr, uint32_t lo, uint32_t hi,
                                            double& Q0, double& g)
{
    while (hi - lo > 1) {
        uint32_t p = pivot(lo, hi);
        if (T.node_r(p) <= tr.r0) lo = p; else hi = p;
    }
    double phi0;
    if (lo == 0) phi0 = __ldg(T.phi);
    else phi0 = __ldg(T.phi + (lo - 1)) - (T.G * __ldg(T.m_cum + (lo - 1))) * (1.0 / tr.r0 - 1.0 / __ldg(T.r + (lo - 1)));
    Q0 = 2.0 * (o.E - phi0) - o.J2 / (tr.r0 * tr.r0);                  // Eq. 12
    g = 0.0;
    if (Q0 > 0.0) g = (o.three_q * (1.0 - tr.s * tr.s)) / sqrt(Q0);
}

// Cold path, reached only if HMC_T_MAX trials were all rejected: redo the star exactly as the
// oracle's loop does, every trial evaluated, remembering the last trial with Q0 > 0.
__device__ __noinline__ void draw_exhaustive(const RTable& T, const Orbit& o, uint32_t seed_lo, uint32_t seed_hi,
                                             uint32_t step, unsigned& st, bool& accepted, uint32_t& used,
                                             bool& have_good, double& good_r, double& good_Q, uint32_t& good_w3)
{
    accepted = false; have_good = false;
    uint32_t t = 0;
    for (; t < HMC_T_MAX; ++t) {
        Trial tr = make_trial(o, seed_lo, seed_hi, step, t);
        double Q0, g;
        exact_trial(T, o, tr, o.kmin, o.kmax + 1, Q0, g);
        if (Q0 > 0.0) {
            have_good = true; good_r = tr.r0; good_Q = Q0; good_w3 = tr.w3;
            if (g > o.F) st |= HMC_STAR_CLIPPED;
            if (o.F * tr.Xp < g) { accepted = true; break; }
        }
    }
    used = accepted ? t + 1 : HMC_T_MAX;
}

__global__ void __launch_bounds__(ORB_THREADS, 1)
sample_new_radius_kernel(uint32_t n, double G, uint32_t seed_lo, uint32_t seed_hi, uint32_t step,
                         const double* __restrict__ r, const double* __restrict__ phi,
                         const double* __restrict__ m_cum, const double* __restrict__ r_mid, int shift,
                         const double* __restrict__ v_r, const double* __restrict__ v_t,
                         const double* __restrict__ E_in, const double* __restrict__ J_in,
                         const double* __restrict__ rmin_in, const double* __restrict__ rmax_in,
                         const uint32_t* __restrict__ kmin_in, const uint32_t* __restrict__ kmax_in,
                         const uint32_t* __restrict__ id, const uint8_t* __restrict__ status_in,
                         double* __restrict__ r_new, double* __restrict__ v_r_new, double* __restrict__ v_t_new,
                         uint16_t* __restrict__ n_try, uint8_t* __restrict__ status_out,
                         unsigned long long* __restrict__ counters)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // coarse[c] = (r, Phi) of node c << shift for 1 <= c <= ncoarse; sentinels (0, Phi_1) and (inf, 0)
    double2* coarse = reinterpret_cast<double2*>(smem_raw);
    const uint32_t ncoarse = n >> shift;
    for (uint32_t c = threadIdx.x + 1; c <= ncoarse; c += ORB_THREADS) {
        uint64_t a = ((uint64_t)c << shift) - 1;
        coarse[c] = make_double2(__ldg(r + a), __ldg(phi + a));
    }
    if (threadIdx.x == 0) { coarse[0] = make_double2(0.0, __ldg(phi)); coarse[ncoarse + 1] = make_double2(pos_inf(), 0.0); }
    __syncthreads();
    RTable T{ r, r_mid, phi, m_cum, G };
    unsigned long long my_trials = 0;

    const uint32_t stride = gridDim.x * ORB_THREADS;
    for (uint32_t a = blockIdx.x * ORB_THREADS + threadIdx.x; a < n; a += stride) {
        unsigned st = status_in[a];
        double out_r = 0.0, out_vr = 0.0, out_vt = 0.0;
        bool moved = false;
        uint32_t used = 0;
        if (!(st & (HMC_STAR_UNBOUND | HMC_STAR_RADIAL | HMC_STAR_DEGENERATE))) {
            Orbit o;
            o.E = __ldcs(E_in + a);
            const double J = __ldcs(J_in + a);
            o.J2 = J * J;
            const double rmin = __ldcs(rmin_in + a), rmax = __ldcs(rmax_in + a);
            o.kmin = __ldcs(kmin_in + a); o.kmax = __ldcs(kmax_in + a);
            const double delta = rmax - rmin;
            bool ok = delta > 0.0;
            o.F = 0.0;
            if (ok) {
                double Bmin = (o.kmin == 0) ? 0.0 : G * __ldg(m_cum + (o.kmin - 1));
                double Bmax = (o.kmax == 0) ? 0.0 : G * __ldg(m_cum + (o.kmax - 1));
                double q1 = (2.0 * (o.J2 / rmin - Bmin)) / (rmin * rmin);      // Q'(r_min) in shell k_min
                double q2 = (2.0 * (o.J2 / rmax - Bmax)) / (rmax * rmax);      // Q'(r_max) in shell k_max
                ok = (q1 > 0.0) && (q2 < 0.0);
                if (ok) o.F = 1.2 * fmax(sqrt((3.0 * delta) / q1), sqrt((3.0 * delta) / (-q2)));
            }
            if (!ok) st |= HMC_STAR_CIRCULAR;
            else {
                o.mid = 0.5 * (rmin + rmax);
                o.quarter = 0.25 * delta; o.three_q = 0.75 * delta;
                o.sid = __ldcs(id + a);
                const uint32_t cl = o.kmin >> shift, ch = o.kmax >> shift;
                bool accepted = false, have_good = false;
                double good_r = 0.0, good_Q = 0.0;
                uint32_t good_w3 = 0, t = 0;
                while (true) {
                    // phase 1: trials decided from shared memory only, until one cannot be rejected
                    Trial tr;
                    uint32_t c = 0;
                    bool cand = false;
                    for (; t < HMC_T_MAX; ++t) {
                        tr = make_trial(o, seed_lo, seed_hi, step, t);
                        uint32_t lo = cl, hi = ch + 1;                 // coarse[lo].x <= r0 < coarse[hi].x (clamped)
                        while (hi - lo > 1) {
                            uint32_t m = (lo + hi) >> 1;
                            if (coarse[m].x <= tr.r0) lo = m; else hi = m;
                        }
                        c = lo;
                        // Phi(r0) lies in [coarse[c].y, coarse[c+1].y]; widen everything by ~1e-11
                        const double u0 = 1.0 / tr.r0;
                        const double cen = (o.J2 * u0) * u0;
                        const double top = 2.0 * (o.E - coarse[c].y);
                        const double tol = 1e-11 * (fabs(top) + cen);
                        const double Qh = (top - cen) + tol;
                        if (Qh <= 0.0) continue;                       // Q0 <= 0 for certain: rejected
                        const double Ql = (2.0 * (o.E - coarse[c + 1].y) - cen) - tol;
                        const double fx = o.F * tr.Xp, cc = o.three_q * (1.0 - tr.s * tr.s);
                        if (Ql > 0.0 && (fx * fx) * Ql > (cc * cc) * (1.0 + 1e-10)) continue;   // F X' > g for certain
                        cand = true;
                        break;
                    }
                    if (!cand) break;
                    // phase 2: the exact test for the candidate
                    const uint32_t lo = max(o.kmin, c << shift);
                    const uint32_t hi = (c >= ncoarse) ? (o.kmax + 1) : min(o.kmax + 1, (c + 1) << shift);
                    double Q0, g;
                    exact_trial(T, o, tr, lo, hi, Q0, g);
                    ++t;
                    if (Q0 > 0.0) {
                        if (g > o.F) st |= HMC_STAR_CLIPPED;
                        if (o.F * tr.Xp < g) {
                            accepted = true; have_good = true; good_r = tr.r0; good_Q = Q0; good_w3 = tr.w3;
                            break;
                        }
                    }
                }
                used = t;
                if (!accepted) draw_exhaustive(T, o, seed_lo, seed_hi, step, st, accepted, used, have_good, good_r, good_Q, good_w3);
                my_trials += used;
                if (!accepted) st |= HMC_STAR_MAXTRIES;
                if (have_good) {
                    moved = true;
                    out_r = good_r;
                    out_vt = J / good_r;
                    double vrn = sqrt(good_Q);                         // v_r = Q^(1/2)
                    out_vr = (good_w3 & 1u) ? -vrn : vrn;
                }
            }
        }
        if (!moved) { out_r = __ldg(r + a); out_vr = __ldcs(v_r + a); out_vt = __ldcs(v_t + a); }
        __stcs(r_new + a, out_r); __stcs(v_r_new + a, out_vr); __stcs(v_t_new + a, out_vt);
        if (n_try) n_try[a] = (uint16_t)used;
        status_out[a] = (uint8_t)st;
        if (counters && (st & (HMC_STAR_CIRCULAR | HMC_STAR_MAXTRIES | HMC_STAR_CLIPPED))) {
            if (st & HMC_STAR_CIRCULAR) atomicAdd(counters + HMC_CNT_CIRCULAR, 1ull);
            if (st & HMC_STAR_MAXTRIES) atomicAdd(counters + HMC_CNT_MAXTRIES, 1ull);
            if (st & HMC_STAR_CLIPPED) atomicAdd(counters + HMC_CNT_CLIPPED, 1ull);
        }
    }
    if (counters) {
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
    const int shift = coarse_shift(n, COARSE_CAP);
    const size_t smem = ((n >> shift) + 2) * sizeof(double2);
    static bool attr_done = false;
    if (!attr_done) {
        HMC_CUDA_TRY(cudaFuncSetAttribute(turning_points_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)(COARSE_CAP * sizeof(double2))));
        attr_done = true;
    }
    int blocks = (int)umin64((n + 255) / 256, (uint64_t)sms * 8);
    build_rphi_kernel<<<blocks, 256, 0, st>>>(r, phi, ws.rphi, ws.rphi_mid, n);
    HMC_LAUNCH_CHECK();
    blocks = (int)umin64((n + ORB_THREADS - 1) / ORB_THREADS, (uint64_t)sms);
    turning_points_kernel<<<blocks, ORB_THREADS, smem, st>>>((uint32_t)n, G, r, v_r, v_t, phi, m_cum, ws.rphi,
                                                            ws.rphi_mid, shift, E, J, r_min, r_max, k_min, k_max, status,
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
    const int sms = sm_count();
    const int shift = coarse_shift(n, COARSE_CAP);
    const size_t smem = ((n >> shift) + 2) * sizeof(double2);
    static bool attr_done = false;
    if (!attr_done) {
        HMC_CUDA_TRY(cudaFuncSetAttribute(sample_new_radius_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)(COARSE_CAP * sizeof(double2))));
        attr_done = true;
    }
    if ((n >> MID_SHIFT) > 0) {
        int blocks = (int)umin64(((n >> MID_SHIFT) + 255) / 256, (uint64_t)sms * 8);
        build_rmid_kernel<<<blocks, 256, 0, st>>>(r, ws.r_mid, n);
        HMC_LAUNCH_CHECK();
    }
    int blocks = (int)umin64((n + ORB_THREADS - 1) / ORB_THREADS, (uint64_t)sms);
    sample_new_radius_kernel<<<blocks, ORB_THREADS, smem, st>>>(
        (uint32_t)n, G, (uint32_t)seed, (uint32_t)(seed >> 32), step, r, phi, m_cum, ws.r_mid, shift, v_r, v_t, E, J,
        r_min, r_max, k_min, k_max, id, status_in, r_new, v_r_new, v_t_new, n_try, status_out,
        reinterpret_cast<unsigned long long*>(counters));
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

}  // namespace hmc
