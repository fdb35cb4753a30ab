// hmc_orbit.cu -- S3 turning points and S4 new-radius draw (Appendix A).
//
// The paper's GPU port ran one thread per star with plain bisection over the (r, Phi) arrays in
// global memory: ~2 log2 N dependent random reads per star for the two
// brackets, and log2 N more per rejection trial.  What is kept: SoA streams for the per-star
// data, one star per thread at a time.  What differs:
//
//  * The bracket predicate "Q(r_j) < 0" is monotone on either side of the star (Q is concave in
//    1/r) and "r_j <= r0" is monotone, so ANY probe order finds the same index.  The searches
//    therefore do not bisect.  They run in three tiers:
//      1. coarse: the nodes that are multiples of S = 2^shift ((r, Phi) pairs, <= 160 KB) are staged
//         once per CTA in shared memory; a bisection over them costs no global traffic and leaves
//         an interval of at most S nodes.
//      2. guess: inside that interval r^2 Q(r) is very nearly linear (the interval spans ~1e-4 of
//         the cluster), so one secant step gives the root radius to a fraction of the node
//         spacing (S3); S4 knows the radius it looks for.  A "radius directory" -- for every coarse
//         interval, S equal-width radius buckets with the offset of the first node of each
//         bucket and of the next, 4 bytes per star, L2 resident up to N = 1e7 -- turns that radius into a
//         node index.
//      3. exact: the node table proper (r_j, Phi_j, G M_j, 1/r_j in one 32-byte sector) is
//         probed at the guess and its neighbour; if the sign change is not there the search
//         gallops away from the guess and bisects what is left.  Typical cost: one directory read
//         and one or two adjacent sectors instead of ~20 dependent probes.
//  * S3 runs the pericentre and the apocentre search of a star interleaved (independent chains).
//  * S4 decides most trials without touching global memory ("squeeze"): Phi is monotone in r, so
//    the shared-memory table brackets Phi(r0) and hence Q(r0) and g; a trial is rejected when the
//    whole bracket, widened by 1e-11, lies on the far side of F X'.  Only the other trials run the
//    exact shell look-up and the exact test, with the oracle's expressions, so the outcome is
//    identical to evaluating every trial.
//  * S4 keeps every lane busy: a lane whose star has been accepted takes the warp's next star at
//    once instead of idling until the slowest of 32 rejection loops ends (the trial count is
//    geometric: mean ~2.5, maximum over a warp ~8).
//  * Random numbers are Philox4x32-10 keyed by (seed, step, star id), not per-thread streams.
#include "hmc_common.cuh"

namespace hmc {

static constexpr int ORB_THREADS = 1024;
static constexpr int ORB_WARPS = ORB_THREADS / 32;
static constexpr int FRONT_ROUNDS = 2;       // S4: trials a lane may run through the squeeze per exact round (1, 3, 4 measured slower)

__device__ __forceinline__ double pos_inf() { return __longlong_as_double(0x7ff0000000000000ll); }

// element of the open interval (lo, hi), hi - lo > 1, with the most trailing zeros
__device__ __forceinline__ uint32_t pivot(uint32_t lo, uint32_t hi)
{
    uint32_t b = hi - 1;
    uint32_t x = lo ^ b;                       // lo < b: highest differing bit is set in b
    int hb = 31 - __clz(x);
    return b & (0xffffffffu << hb);
}

__device__ __forceinline__ Node ld_node(const Node* __restrict__ p)
{
    Node e;
    // L1::no_allocate: with ~200 KB of the SM's 256 KB carved out as shared memory the L1 is tiny, and
    // random sector loads that allocate in it run at half the rate of loads that bypass it
    // (measured: 126 vs 263 random 32-byte loads per ns from an L2-resident table).
    asm("ld.global.nc.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(e.r), "=d"(e.phi), "=d"(e.B), "=d"(e.u) : "l"(p));
    return e;
}

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

__device__ __forceinline__ double2 ld_d2_na(const double2* __restrict__ p)
{
    double2 v;
    asm("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}

__device__ __forceinline__ uint32_t ld_u32_na(const uint32_t* __restrict__ p)
{
    uint32_t v;
    asm("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}

// The radius directory (4 bytes per star) is small enough to live in the 126 MB L2, the node table
// (32 bytes per star) is not, and every star reads a few random lines of each: directory lines are
// loaded with an evict-last L2 policy so that the node traffic streaming through L2 does not push them out.
__device__ __forceinline__ uint64_t l2_keep_policy()
{
    uint64_t pol;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}

__device__ __forceinline__ uint32_t ld_u32_keep(const uint32_t* __restrict__ p, uint64_t pol)
{
    uint32_t v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.u32 %0, [%1], %2;" : "=r"(v) : "l"(p), "l"(pol));
    return v;
}

// ---- radius directory -------------------------------------------------------------------------
// Coarse interval c holds the nodes j with j >> shift == c (j >= 1); its radii lie in [Rl, Rh],
// Rl = r of node c << shift (0 for c = 0), Rh = r of node (c+1) << shift (r_N in the last
// interval).  bucket() maps a radius of the interval to one of K = 2^shift equal-width buckets;
// it is monotone non-decreasing in x, which is all the look-up relies on.  With o_b = number of
// nodes of the interval whose bucket is < b (b = 0..K), entry b of the interval's row is the
// 32-bit word o_b | o_{b+1} << 16, b = 0..K-1: one load gives both ends of a bucket.
__device__ __forceinline__ float bucket_scale(double Rl, double Rh, uint32_t K) { return (float)K / (float)(Rh - Rl); }

__device__ __forceinline__ uint32_t bucket(double x, double Rl, float scale, uint32_t K)
{
    float t = (float)(x - Rl) * scale;
    uint32_t b = 0;                                        // t < 0 or NaN (Rh == Rl)
    if (t >= 0.0f) b = (t < (float)K) ? (uint32_t)t : K - 1;
    return b;
}

// nodes[j], j = 0..n+1
__global__ void __launch_bounds__(256) build_nodes_kernel(const double* __restrict__ r, const double* __restrict__ phi,
                                                          const double* __restrict__ m_cum, double G,
                                                          Node* __restrict__ nodes, double2* __restrict__ coarse_g,
                                                          double2* __restrict__ mid_g, int shift, uint64_t n,
                                                          uint32_t* __restrict__ s4_words)
{
    if (blockIdx.x == 0 && threadIdx.x == 0) { s4_words[0] = 0; s4_words[1] = 0; }      // S4's batch and exit counters
    const uint64_t low_mask = (1ull << shift) - 1;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; j <= n + 1; j += stride) {
        Node e;
        if (j == 0) { e.r = 0.0; e.phi = __ldg(phi); e.B = 0.0; e.u = 0.0; }
        else if (j == n + 1) { e.r = pos_inf(); e.phi = 0.0; e.B = G * __ldg(m_cum + (n - 1)); e.u = 0.0; }
        else {
            const double rj = __ldcs(r + (j - 1));
            e.r = rj; e.phi = __ldcs(phi + (j - 1)); e.B = G * __ldcs(m_cum + (j - 1)); e.u = 1.0 / rj;
        }
        nodes[j] = e;
        if ((j & low_mask) == 0 && j <= n) coarse_g[j >> shift] = make_double2(e.r, e.phi);
        if (shift > MID_SHIFT && (j & ((1u << MID_SHIFT) - 1)) == 0 && j <= n) mid_g[j >> MID_SHIFT] = make_double2(e.r, e.phi);
    }
}

// The tables of one coarse interval, by one CTA (shift > 0): the interval's nodes are written (r, Phi, M read once,
// coalesced), counted into their buckets in shared memory (radii ascend, so neighbouring threads hit neighbouring
// counters), the counts are scanned, and the directory row is written as whole 32-bit entries, coalesced.
// The CTA of interval 0 also writes the sentinel node 0, the last one node N+1; coarse and mid entries are written
// by whoever owns the node.
static constexpr int DIR_THREADS = 256;

__global__ void __launch_bounds__(DIR_THREADS) build_tables_kernel(const double* __restrict__ r, const double* __restrict__ phi,
                                                                   const double* __restrict__ m_cum, double G,
                                                                   Node* __restrict__ nodes, double2* __restrict__ coarse_g,
                                                                   double2* __restrict__ mid_g, uint32_t* __restrict__ dir,
                                                                   uint32_t n, int shift, uint32_t* __restrict__ s4_words)
{
    if (blockIdx.x == 0 && threadIdx.x == 0) { s4_words[0] = 0; s4_words[1] = 0; }      // S4's batch and exit counters
    extern __shared__ uint32_t cnt[];                                // [K + 1]: cnt[b + 1] = nodes in bucket b, then o_b
    __shared__ uint32_t warp_tot[DIR_THREADS / 32];
    const uint32_t K = 1u << shift, c = blockIdx.x;
    const uint32_t j0 = max(c << shift, 1u);                         // first node of the interval
    const uint32_t jn = min(((c + 1) << shift) - 1, n);              // last node of the interval
    const double Rl = c ? __ldg(r + ((c << shift) - 1)) : 0.0;
    const double Rh = (((uint64_t)(c + 1) << shift) <= n) ? __ldg(r + (((c + 1) << shift) - 1)) : __ldg(r + (n - 1));
    const float scale = bucket_scale(Rl, Rh, K);
    for (uint32_t b = threadIdx.x; b <= K; b += DIR_THREADS) cnt[b] = 0;
    if (threadIdx.x == 0) {
        if (c == 0) {
            Node e; e.r = 0.0; e.phi = __ldg(phi); e.B = 0.0; e.u = 0.0;
            nodes[0] = e;
            coarse_g[0] = make_double2(e.r, e.phi);
            if (shift > MID_SHIFT) mid_g[0] = make_double2(e.r, e.phi);
        }
        if (c == gridDim.x - 1) {
            Node e; e.r = pos_inf(); e.phi = 0.0; e.B = G * __ldg(m_cum + (n - 1)); e.u = 0.0;
            nodes[(size_t)n + 1] = e;
        }
    }
    __syncthreads();
    const uint32_t low_mask = K - 1u;
    for (uint32_t j = j0 + threadIdx.x; j <= jn; j += DIR_THREADS) {
        Node e;
        const double rj = __ldcs(r + (j - 1));
        e.r = rj; e.phi = __ldcs(phi + (j - 1)); e.B = G * __ldcs(m_cum + (j - 1)); e.u = 1.0 / rj;
        nodes[j] = e;
        if ((j & low_mask) == 0) coarse_g[j >> shift] = make_double2(e.r, e.phi);
        if (shift > MID_SHIFT && (j & ((1u << MID_SHIFT) - 1)) == 0) mid_g[j >> MID_SHIFT] = make_double2(e.r, e.phi);
        atomicAdd(&cnt[bucket(rj, Rl, scale, K) + 1], 1u);
    }
    __syncthreads();
    // inclusive scan of cnt[0 .. K] in place: cnt[b] becomes o_b = number of nodes with bucket < b
    const uint32_t per = (K + 1 + DIR_THREADS - 1) / DIR_THREADS;
    const uint32_t b0 = min(K + 1, threadIdx.x * per), b1 = min(K + 1, b0 + per);
    uint32_t sum = 0;
    for (uint32_t b = b0; b < b1; ++b) sum += cnt[b];
    uint32_t inc = sum;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    uint32_t run = inc - sum;
    for (uint32_t w = 0; w < warp; ++w) run += warp_tot[w];
    for (uint32_t b = b0; b < b1; ++b) { run += cnt[b]; cnt[b] = run; }
    __syncthreads();
    uint32_t* row = dir + (size_t)c * K;
    for (uint32_t b = threadIdx.x; b < K; b += DIR_THREADS) row[b] = cnt[b] | (cnt[b + 1] << 16);
}

// The same for narrow intervals (K = 2^shift <= 256 nodes: N below about 2.6e6): one WARP per interval, eight
// intervals per CTA, no block-wide barrier.  (One CTA per interval left most of its 256 threads without a node:
// 27 us at N = 1e6, where the whole turning-point stage takes 100 us.)
static constexpr int DIR_SMALL_MAX_K = 256;

__global__ void __launch_bounds__(DIR_THREADS) build_tables_small_kernel(const double* __restrict__ r, const double* __restrict__ phi,
                                                                         const double* __restrict__ m_cum, double G,
                                                                         Node* __restrict__ nodes, double2* __restrict__ coarse_g,
                                                                         uint32_t* __restrict__ dir, uint32_t n, int shift,
                                                                         uint32_t nintervals, uint32_t* __restrict__ s4_words)
{
    __shared__ uint32_t cnt_all[DIR_THREADS / 32][DIR_SMALL_MAX_K + 1];
    if (blockIdx.x == 0 && threadIdx.x == 0) { s4_words[0] = 0; s4_words[1] = 0; }      // S4's batch and exit counters
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t K = 1u << shift, c = blockIdx.x * (DIR_THREADS / 32) + warp;
    if (c >= nintervals) return;
    uint32_t* cnt = cnt_all[warp];
    const uint32_t j0 = max(c << shift, 1u), jn = min(((c + 1) << shift) - 1, n);
    const double Rl = c ? __ldg(r + ((c << shift) - 1)) : 0.0;
    const double Rh = (((uint64_t)(c + 1) << shift) <= n) ? __ldg(r + (((c + 1) << shift) - 1)) : __ldg(r + (n - 1));
    const float scale = bucket_scale(Rl, Rh, K);
    for (uint32_t b = lane; b <= K; b += 32) cnt[b] = 0;
    if (lane == 0) {
        if (c == 0) {
            Node e; e.r = 0.0; e.phi = __ldg(phi); e.B = 0.0; e.u = 0.0;
            nodes[0] = e;
            coarse_g[0] = make_double2(e.r, e.phi);
        }
        if (c == nintervals - 1) {
            Node e; e.r = pos_inf(); e.phi = 0.0; e.B = G * __ldg(m_cum + (n - 1)); e.u = 0.0;
            nodes[(size_t)n + 1] = e;
        }
    }
    __syncwarp();
    for (uint32_t j = j0 + lane; j <= jn; j += 32) {
        Node e;
        const double rj = __ldcs(r + (j - 1));
        e.r = rj; e.phi = __ldcs(phi + (j - 1)); e.B = G * __ldcs(m_cum + (j - 1)); e.u = 1.0 / rj;
        nodes[j] = e;
        if ((j & (K - 1u)) == 0) coarse_g[j >> shift] = make_double2(e.r, e.phi);
        atomicAdd(&cnt[bucket(rj, Rl, scale, K) + 1], 1u);
    }
    __syncwarp();
    // inclusive scan of cnt[0 .. K] in place: cnt[b] becomes o_b = number of nodes with bucket < b
    const uint32_t per = (K + 1 + 31) / 32;
    const uint32_t b0 = min(K + 1, lane * per), b1 = min(K + 1, b0 + per);
    uint32_t sum = 0;
    for (uint32_t b = b0; b < b1; ++b) sum += cnt[b];
    uint32_t inc = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
    uint32_t run = inc - sum;
    for (uint32_t b = b0; b < b1; ++b) { run += cnt[b]; cnt[b] = run; }
    __syncwarp();
    uint32_t* row = dir + (size_t)c * K;
    for (uint32_t b = lane; b < K; b += 32) row[b] = cnt[b] | (cnt[b + 1] << 16);
}

// coarse[c] = (r, Phi) of node c << shift, c = 1..ncoarse; coarse[0] = (0, Phi_1) and
// coarse[ncoarse + 1] = (+inf, 0) are the sentinel nodes 0 and N+1.
__device__ __forceinline__ void stage_coarse(double2* coarse, const double2* __restrict__ coarse_g, uint32_t n, int shift)
{
    const uint32_t ncoarse = n >> shift;
    for (uint32_t c = threadIdx.x; c <= ncoarse; c += ORB_THREADS) coarse[c] = __ldg(coarse_g + c);
    if (threadIdx.x == 0) coarse[ncoarse + 1] = make_double2(pos_inf(), 0.0);
    __syncthreads();
}

// Radii of the coarse nodes in shared memory: either the x components of the (r, Phi) pairs (step 2 doubles) or, in
// the sampler, an array of their own (step 1; Phi is kept beside it as binary32, see sample_new_radius_kernel).
struct CoarseR {
    const double* p;
    int sh;                  // log2 of the step in doubles
    __device__ __forceinline__ double operator[](uint32_t c) const { return p[(size_t)c << sh]; }
};

struct Tables {
    const Node* nodes;       // [n + 2]
    const uint32_t* dir;
    const double2* coarse;   // shared memory: (r, Phi) pairs, or nullptr when only the radii are there (cr)
    const double2* mid;      // global (L2): (r, Phi) of every 2^MID_SHIFT-th node when shift > MID_SHIFT, else nullptr
    double r_last;           // r_N
    uint32_t n, ncoarse, K;
    int shift;
    uint64_t keep;           // L2 evict-last policy for directory loads
    CoarseR cr;              // radii of the coarse nodes
    // (r, Phi) of node j, j a multiple of the finest table spacing in use
    __device__ __forceinline__ double2 aligned_node(uint32_t j) const { return mid ? ld_d2_na(mid + (j >> MID_SHIFT)) : coarse[j >> shift]; }
    // upper radius of coarse interval c, as build_dir_kernel defines it
    __device__ __forceinline__ double interval_rh(uint32_t c) const { return c < ncoarse ? cr[c + 1] : r_last; }
    // nodes lo < hi with  r_lo <= x < r_hi  as far as the directory knows: every node of interval c
    // outside (lo, hi) is on the side stated.  x must lie in the radius range of interval c for the
    // result to be tight; for any x it is a valid starting point of an exact search.
    __device__ __forceinline__ void dir_range(uint32_t c, double x, uint32_t& lo, uint32_t& hi) const
    {
        const double Rl = cr[c];
        const uint32_t b = bucket(x, Rl, bucket_scale(Rl, interval_rh(c), K), K);
        const uint32_t w = ld_u32_keep(dir + (size_t)c * K + b, keep);
        const uint32_t o0 = w & 0xffffu, o1 = w >> 16;
        const uint32_t j0 = max(c << shift, 1u);
        lo = j0 + o0 - 1;
        hi = j0 + o1;
    }
    // Most likely last node at or below x: the nodes strictly inside dir_range's (lo, hi) share x's
    // bucket, and about the fraction of the bucket that lies below x of them are below x.  A guess only.
    // In two halves, so that a caller with two radii can have both directory loads in flight at once.
    __device__ __forceinline__ const uint32_t* dir_guess_slot(uint32_t c, double x, float& frac) const
    {
        const double Rl = cr[c];
        const float scale = bucket_scale(Rl, interval_rh(c), K);
        const uint32_t b = bucket(x, Rl, scale, K);
        frac = fminf(fmaxf((float)(x - Rl) * scale - (float)b, 0.0f), 1.0f);
        return dir + (size_t)c * K + b;
    }
    __device__ __forceinline__ uint32_t dir_guess_node(uint32_t c, uint32_t w, float frac) const
    {
        const uint32_t o0 = w & 0xffffu, o1 = w >> 16;
        return max(c << shift, 1u) + o0 - 1 + (uint32_t)(frac * (float)(o1 - o0) + 0.5f);
    }
};

// ---- S3 ---------------------------------------------------------------------------------------
// Q(r_p) < 0, division-free (R2):  2 (E - Phi_p) r_p^2 < J^2
__device__ __forceinline__ bool q_negative(double rp, double phip, double E, double J2)
{
    return 2.0 * ((E - phip) * (rp * rp)) < J2;
}

// One side of the bracket search after the coarse tier.  The invariant is: node lo is "inside the
// class" (pericentre: Q < 0; apocentre: Q >= 0), node hi is not; done when hi - lo == 1.
enum { MODE_GUESS = 0, MODE_UP = 1, MODE_DOWN = 2, MODE_BISECT = 3 };

struct Side {
    uint32_t lo, hi, step, guess;
    int mode;
    __device__ __forceinline__ bool active() const { return hi - lo > 1; }
    // first node of the adjacent pair (p, p+1) to probe next; lo < p < hi
    __device__ __forceinline__ uint32_t probe() const
    {
        uint32_t p;
        if (mode == MODE_GUESS) p = guess;
        else if (mode == MODE_UP) p = lo + step;
        else if (mode == MODE_DOWN) p = (hi > step + 1) ? hi - step - 1 : 0;
        else p = lo + (hi - lo) / 2;
        return min(max(p, lo + 1), hi - 1);
    }
    // c0 / c1: node p / p+1 is inside the class (c1 is ignored when p + 1 == hi)
    __device__ __forceinline__ void update(uint32_t p, bool c0, bool c1)
    {
        const bool two = p + 1 < hi;
        if (two && c1) {                       // both inside: the sign change is above p+1
            lo = p + 1;
            if (mode == MODE_GUESS) { mode = MODE_UP; step = 1; }
            else if (mode == MODE_UP) step *= 2;
            else mode = MODE_BISECT;
        } else if (c0) {                       // p inside, p+1 outside (or p+1 == hi)
            lo = p;
            if (two) hi = p + 1;
            mode = MODE_BISECT;
        } else {                               // p outside: the sign change is below p
            hi = p;
            if (mode == MODE_GUESS) { mode = MODE_DOWN; step = 1; }
            else if (mode == MODE_DOWN) step *= 2;
            else mode = MODE_BISECT;
        }
    }
};

// Secant estimate of the root of P(r) = r^2 Q(r) between two nodes with P_lo and P_hi of opposite
// sign; the directory turns it into a node number.  Only a starting point: any value works.
__device__ __forceinline__ double secant_root(double r_lo, double P_lo, double r_hi, double P_hi)
{
    return r_lo + (r_hi - r_lo) * (P_lo / (P_lo - P_hi));
}

// One star of S3: brackets, turning points, status, and S4's bound F (0 = no draw).  a = position in the
// sorted arrays (star k = a + 1); rk, vr, vt, phik its radius, velocities and potential.  In two halves:
// locate_star (tiers 1 and 2: shared memory and the directory, ends with the guessed nodes) and finish_star_s3
// (tier 3: the exact probes, then the roots), so that a caller can put other work between the two while the
// guessed nodes travel from DRAM to L2.
struct Solved {
    double E, J, rmin, rmax, Fv;
    uint32_t kmin, kmax;
    unsigned st;
};

struct Located {
    double E, J, rk;
    uint32_t lo1, hi1, g1, lo2, hi2, g2;   // brackets after tiers 1-2 and the guessed nodes (pericentre 1, apocentre 2)
    unsigned st;                            // status bits; bit 8 / bit 9: side 1 / 2 starts from its guess
};

__device__ __forceinline__ Located locate_star(const Tables& T, uint32_t a, double rk, double vr, double vt, double phik)
{
    const uint32_t n = T.n;
    const int shift = T.shift;
    const double2* coarse = T.coarse;
    const uint32_t k = a + 1;
    Located L;
    const double E = phik + 0.5 * (vr * vr + vt * vt);      // Eq. 16
    const double J = rk * vt;
    const double J2 = J * J;
    unsigned st = 0;
    if (!(E < 0.0)) st |= HMC_STAR_UNBOUND;
    if (J2 == 0.0) st |= HMC_STAR_RADIAL;
    L.E = E; L.J = J; L.rk = rk;
    L.lo1 = 0u; L.hi1 = k; L.g1 = 0u; L.lo2 = k; L.hi2 = n + 1; L.g2 = 0u;
    if (!st) {
        // pericentre bracket (lo, hi): Q_lo < 0 <= Q_hi;  apocentre: Q_lo >= 0 > Q_hi
        Side s1{ 0u, k, 1u, 0u, MODE_BISECT }, s2{ k, n + 1, 1u, 0u, MODE_BISECT };
        // tier 1: the coarse nodes, in shared memory; both searches advance together (two
        // independent chains of dependent shared-memory loads instead of one after the other).
        // Pericentre: largest coarse c in [0, ck] with Q < 0 (c = 0 is node 0, always < 0).
        // Apocentre: smallest coarse c in [cka, ncoarse + 1] with Q < 0 (ncoarse + 1 stands for node N+1).
        {
            const uint32_t ck = (k - 1) >> shift, cka = (k >> shift) + 1;
            uint32_t l1 = 0, h1 = ck + 1, l2 = cka - 1, h2 = T.ncoarse + 1;
            while (true) {
                const bool a1 = h1 - l1 > 1, a2 = h2 - l2 > 1;
                if (!(a1 || a2)) break;
                const uint32_t m1 = (l1 + h1) >> 1, m2 = (l2 + h2) >> 1;
                const double2 e1 = coarse[a1 ? m1 : 0u], e2 = coarse[a2 ? m2 : 0u];
                const bool n1 = q_negative(e1.x, e1.y, E, J2), n2 = q_negative(e2.x, e2.y, E, J2);
                l1 = (a1 && n1) ? m1 : l1; h1 = (a1 && !n1) ? m1 : h1;
                h2 = (a2 && n2) ? m2 : h2; l2 = (a2 && !n2) ? m2 : l2;
            }
            s1.lo = l1 << shift; s1.hi = (l1 == ck) ? k : ((l1 + 1) << shift);
            s2.hi = (h2 <= T.ncoarse) ? (h2 << shift) : n + 1; s2.lo = (h2 == cka) ? k : ((h2 - 1) << shift);
        }
        // tier 1b (large N only, shift > MID_SHIFT): a coarse interval then holds 2^shift >> 1024 nodes and
        // r^2 Q is no longer linear across it; bisect on over every 1024-th node, a table small
        // enough to stay in L2, both sides together.
        if (T.mid) {
            uint32_t l1 = s1.lo >> MID_SHIFT, h1 = (s1.hi + ((1u << MID_SHIFT) - 1)) >> MID_SHIFT;
            uint32_t l2 = s2.lo >> MID_SHIFT, h2 = (s2.hi > n) ? (n >> MID_SHIFT) + 1 : (s2.hi >> MID_SHIFT);
            while (true) {
                const bool a1 = h1 - l1 > 1, a2 = h2 - l2 > 1;
                if (!(a1 || a2)) break;
                const uint32_t m1 = (l1 + h1) >> 1, m2 = (l2 + h2) >> 1;
                const double2 e1 = ld_d2_na(T.mid + (a1 ? m1 : 0u)), e2 = ld_d2_na(T.mid + (a2 ? m2 : 0u));
                const bool n1 = q_negative(e1.x, e1.y, E, J2), n2 = q_negative(e2.x, e2.y, E, J2);
                l1 = (a1 && n1) ? m1 : l1; h1 = (a1 && !n1) ? m1 : h1;
                h2 = (a2 && n2) ? m2 : h2; l2 = (a2 && !n2) ? m2 : l2;
            }
            s1.lo = max(s1.lo, l1 << MID_SHIFT); s1.hi = min(s1.hi, h1 << MID_SHIFT);
            s2.lo = max(s2.lo, l2 << MID_SHIFT); if (h2 <= (n >> MID_SHIFT)) s2.hi = min(s2.hi, h2 << MID_SHIFT);
        }
        // tier 2: secant guess.  The ends are table nodes or the star's own node, where
        // P = r^2 Q = (r_k v_r)^2.  The first and last intervals (a sentinel at one end) bisect.
        const double Pk = (rk * vr) * (rk * vr);
        const bool g1 = s1.hi - s1.lo > 2 && s1.lo > 0, g2 = s2.hi - s2.lo > 2 && s2.hi <= n;
        double x1 = 0.0, x2 = 0.0;
        if (g1) {
            double2 el = T.aligned_node(s1.lo);
            double r_hi = rk, P_hi = Pk;
            if (s1.hi != k) { double2 eh = T.aligned_node(s1.hi); r_hi = eh.x; P_hi = 2.0 * ((E - eh.y) * (eh.x * eh.x)) - J2; }
            x1 = secant_root(el.x, 2.0 * ((E - el.y) * (el.x * el.x)) - J2, r_hi, P_hi);
        }
        if (g2) {
            double2 eh = T.aligned_node(s2.hi);
            double r_lo = rk, P_lo = Pk;
            if (s2.lo != k) { double2 el = T.aligned_node(s2.lo); r_lo = el.x; P_lo = 2.0 * ((E - el.y) * (el.x * el.x)) - J2; }
            x2 = secant_root(r_lo, P_lo, eh.x, 2.0 * ((E - eh.y) * (eh.x * eh.x)) - J2);
        }
        {   // both directory entries in flight together
            float f1 = 0.0f, f2 = 0.0f;
            const uint32_t c1 = s1.lo >> shift, c2 = s2.lo >> shift;
            const uint32_t* a1 = g1 ? T.dir_guess_slot(c1, x1, f1) : nullptr;
            const uint32_t* a2 = g2 ? T.dir_guess_slot(c2, x2, f2) : nullptr;
            uint32_t w1 = 0, w2 = 0;
            if (g1) w1 = ld_u32_keep(a1, T.keep);
            if (g2) w2 = ld_u32_keep(a2, T.keep);
            if (g1) { s1.guess = T.dir_guess_node(c1, w1, f1); st |= 256u; }
            if (g2) { s2.guess = T.dir_guess_node(c2, w2, f2); st |= 512u; }
        }
        L.lo1 = s1.lo; L.hi1 = s1.hi; L.g1 = s1.guess; L.lo2 = s2.lo; L.hi2 = s2.hi; L.g2 = s2.guess;
    }
    L.st = st;
    return L;
}

// Tier 3 by lane pairs (warp-collective: all 32 lanes call it together; a lane without a search passes closed
// sides).  What a random access to a table of gigabytes costs is the REQUEST -- one per load instruction and
// 128-byte line, about 37 per ns on the whole chip once the table is far beyond the reach of the TLB -- not the
// bytes (profiles/r2_random_access.md).  A lane that loads nodes p and p+1 itself issues two instructions, hence two requests,
// and a third to fetch the bracketing node again for the roots.  Here lanes 2i and 2i+1 serve their two stars one
// after the other: for the star whose turn it is, the even lane loads node p and the odd lane node p+1 in the SAME
// instruction (one request when both lie in one line, 3 times in 4), each evaluates the sign of Q at its node for
// that star, the answers come back in a ballot, and when a side closes the lane that holds the bracketing node
// hands it over through shuffles.  Same probes, same brackets as the one-lane search.
__device__ __forceinline__ Node shfl_node(const Node& e, int src)
{
    Node t;
    t.r = __shfl_sync(0xffffffffu, e.r, src); t.phi = __shfl_sync(0xffffffffu, e.phi, src);
    t.B = __shfl_sync(0xffffffffu, e.B, src); t.u = __shfl_sync(0xffffffffu, e.u, src);
    return t;
}

// keep1 / keep2: the bracketing node of side 1 / 2 when have1 / have2 (else the caller loads it).
// (Handing the nodes over through 64 KB of shared memory instead of shuffles is 1-5 % faster where the coarse table
// is small -- 15.8 against 16.0 ms at N = 1e8 -- and 70 % slower where it takes its full 160 KB, e.g. N = 4.19e7:
// 10.7 against 6.3 ms, one lane per star 6.9: nothing is left of the L1 then.)
__device__ __forceinline__ void probe_pairs(const Node* __restrict__ nodes, Side& s1, Side& s2, double E, double J2,
                                            Node& keep1, Node& keep2, bool& have1, bool& have2, uint32_t lane)
{
    have1 = have2 = false;
    const uint32_t odd = lane & 1u, even_lane = lane & ~1u;
    while (true) {
        const bool a1 = s1.active(), a2 = s2.active();
        if (!__any_sync(0xffffffffu, a1 || a2)) break;
        const uint32_t p1 = a1 ? s1.probe() : 0u, p2 = a2 ? s2.probe() : 0u;
        const uint32_t act = (a1 ? 1u : 0u) | (a2 ? 2u : 0u);
#pragma unroll
        for (int h = 0; h < 2; ++h) {                          // h: whose star the pair serves
            const int owner = (int)(even_lane | (uint32_t)h);
            const bool own = odd == (uint32_t)h;
            const uint32_t P1 = __shfl_sync(0xffffffffu, p1, owner), P2 = __shfl_sync(0xffffffffu, p2, owner);
            const uint32_t A = __shfl_sync(0xffffffffu, act, owner);
            const double Eo = __shfl_sync(0xffffffffu, E, owner), J2o = __shfl_sync(0xffffffffu, J2, owner);
            Node n1{ 0.0, 0.0, 0.0, 0.0 }, n2{ 0.0, 0.0, 0.0, 0.0 };
            bool neg1 = false, neg2 = false;
            if (A & 1u) { n1 = ld_node(nodes + P1 + odd); neg1 = q_negative(n1.r, n1.phi, Eo, J2o); }
            if (A & 2u) { n2 = ld_node(nodes + P2 + odd); neg2 = q_negative(n2.r, n2.phi, Eo, J2o); }
            const unsigned b1 = __ballot_sync(0xffffffffu, neg1), b2 = __ballot_sync(0xffffffffu, neg2);
            // the owner moves its brackets; a side that closes on a node of this probe names the lane holding it
            uint32_t want = 0;                                  // bits 0-1 side 1, bits 2-3 side 2: 1 = even lane, 2 = odd lane
            if (own) {
                if (a1) {
                    s1.update(p1, ((b1 >> even_lane) & 1u) != 0u, ((b1 >> (even_lane + 1u)) & 1u) != 0u);
                    if (!s1.active()) want |= (s1.lo == p1) ? 1u : ((s1.lo == p1 + 1u) ? 2u : 0u);
                }
                if (a2) {
                    s2.update(p2, ((b2 >> even_lane) & 1u) == 0u, ((b2 >> (even_lane + 1u)) & 1u) == 0u);
                    if (!s2.active()) want |= (s2.lo == p2) ? 4u : ((s2.lo == p2 + 1u) ? 8u : 0u);
                }
                have1 = have1 || (want & 3u); have2 = have2 || (want & 12u);
            }
            const uint32_t W = __shfl_sync(0xffffffffu, want, owner);
            if (__any_sync(0xffffffffu, (W & 3u) != 0u)) {      // some pair closed side 1 on a node of this probe
                const Node t = shfl_node(n1, (int)(even_lane | ((W & 2u) ? 1u : 0u)));
                if (own && (W & 3u)) keep1 = t;
            }
            if (__any_sync(0xffffffffu, (W & 12u) != 0u)) {
                const Node t = shfl_node(n2, (int)(even_lane | ((W & 8u) ? 1u : 0u)));
                if (own && (W & 12u)) keep2 = t;
            }
        }
    }
}

// Closed-form roots of Q(u) = 2C + 2Bu - J^2 u^2 in the bracketing shells (R3), from their nodes ea (shell k_min) and
// eb (shell k_max); sets DEGENERATE when the outer quadratic has C >= 0.  Shared by the one-lane and the lane-pair search.
__device__ __forceinline__ void roots_and_bound(const Node ea, const Node eb, double E, double J2, double& rmin, double& rmax,
                                                double& Fv, unsigned& st)
{
    const double Ca = (E - ea.phi) - ea.B * ea.u;
    const double Cb = (E - eb.phi) - eb.B * eb.u;
    double D = ea.B * ea.B + 2.0 * (J2 * Ca);
    if (D < 0.0) D = 0.0;
    rmin = J2 / (ea.B + sqrt(D));
    D = eb.B * eb.B + 2.0 * (J2 * Cb);
    if (D < 0.0) D = 0.0;
    if (Cb < 0.0) rmax = (eb.B + sqrt(D)) / (-2.0 * Cb);
    else { rmax = pos_inf(); st |= HMC_STAR_DEGENERATE; }
    // S4's bound F (R7) needs G M at both bracketing shells, which are in registers here and
    // would cost S4 two random node reads per star: computed here and left in the workspace for a
    // following S4 call with reuse_tables (0 = no draw).  S4 writes F = 1.2 max(sqrt(3 D / q1), sqrt(3 D / -q2));
    // division and square root are correctly rounded, hence monotone, so the larger square root is the
    // square root of the larger quotient, which is the quotient by the smaller divisor: the same bits
    // from one division and one square root instead of two each.
    const double delta = rmax - rmin;
    if (!(st & HMC_STAR_DEGENERATE) && delta > 0.0) {
        const double q1 = (2.0 * (J2 / rmin - ea.B)) / (rmin * rmin);      // Q'(r_min) in shell k_min
        const double q2 = (2.0 * (J2 / rmax - eb.B)) / (rmax * rmax);      // Q'(r_max) in shell k_max
        if ((q1 > 0.0) && (q2 < 0.0)) Fv = 1.2 * sqrt((3.0 * delta) / fmin(q1, -q2));
    }
}

__device__ __forceinline__ Solved finish_star_s3(const Tables& T, uint32_t a, const Located& L)
{
    const Node* __restrict__ nodes = T.nodes;
    const uint32_t k = a + 1;
    const double E = L.E, J = L.J, rk = L.rk, J2 = J * J;
    double rmin, rmax, Fv = 0.0;
    uint32_t kmin, kmax;
    unsigned st = L.st & 255u;
    if (st) {
        rmin = (st & HMC_STAR_RADIAL) ? 0.0 : rk;
        rmax = (st & HMC_STAR_UNBOUND) ? pos_inf() : rk;
        kmin = k - 1; kmax = k;
    } else {
        Side s1{ L.lo1, L.hi1, 1u, L.g1, (L.st & 256u) ? MODE_GUESS : MODE_BISECT }, s2{ L.lo2, L.hi2, 1u, L.g2, (L.st & 512u) ? MODE_GUESS : MODE_BISECT };
        // tier 3: exact probes of adjacent node pairs, the two searches interleaved
        while (true) {
            const bool a1 = s1.active(), a2 = s2.active();
            if (!(a1 || a2)) break;
            const uint32_t p1 = a1 ? s1.probe() : 0u, p2 = a2 ? s2.probe() : 0u;
            Node e10, e11, e20, e21;
            if (a1) { e10 = ld_node(nodes + p1); e11 = ld_node(nodes + p1 + 1); }
            if (a2) { e20 = ld_node(nodes + p2); e21 = ld_node(nodes + p2 + 1); }
            if (a1) s1.update(p1, q_negative(e10.r, e10.phi, E, J2), q_negative(e11.r, e11.phi, E, J2));
            if (a2) s2.update(p2, !q_negative(e20.r, e20.phi, E, J2), !q_negative(e21.r, e21.phi, E, J2));
        }
        kmin = s1.lo; kmax = s2.lo;
        roots_and_bound(ld_node(nodes + kmin), ld_node(nodes + kmax), E, J2, rmin, rmax, Fv, st);
    }
    return Solved{ E, J, rmin, rmax, Fv, kmin, kmax, st };
}

// The same with tier 3 by lane pairs: the whole warp must call this together, `valid` false for a lane without a star.
__device__ __forceinline__ Solved finish_star_s3_pairs(const Tables& T, uint32_t a, const Located& L, bool valid, uint32_t lane)
{
    const Node* __restrict__ nodes = T.nodes;
    const uint32_t k = a + 1;
    const double E = L.E, J = L.J, rk = L.rk, J2 = J * J;
    double rmin = rk, rmax = rk, Fv = 0.0;
    uint32_t kmin = k - 1, kmax = k;
    unsigned st = L.st & 255u;
    const bool search = valid && !st;
    Side s1{ L.lo1, L.hi1, 1u, L.g1, (L.st & 256u) ? MODE_GUESS : MODE_BISECT }, s2{ L.lo2, L.hi2, 1u, L.g2, (L.st & 512u) ? MODE_GUESS : MODE_BISECT };
    if (!search) { s1.lo = 0u; s1.hi = 1u; s2.lo = 0u; s2.hi = 1u; }           // closed
    bool have_a = false, have_b = false;
    Node ka{ 0.0, 0.0, 0.0, 0.0 }, kb{ 0.0, 0.0, 0.0, 0.0 };
    probe_pairs(nodes, s1, s2, E, J2, ka, kb, have_a, have_b, lane);
    if (st) {
        rmin = (st & HMC_STAR_RADIAL) ? 0.0 : rk;
        rmax = (st & HMC_STAR_UNBOUND) ? pos_inf() : rk;
    } else if (valid) {
        kmin = s1.lo; kmax = s2.lo;
        roots_and_bound(have_a ? ka : ld_node(nodes + kmin), have_b ? kb : ld_node(nodes + kmax), E, J2, rmin, rmax, Fv, st);
    }
    return Solved{ E, J, rmin, rmax, Fv, kmin, kmax, st };
}

__device__ __forceinline__ Solved solve_star(const Tables& T, uint32_t a, double rk, double vr, double vt, double phik)
{
    return finish_star_s3(T, a, locate_star(T, a, rk, vr, vt, phik));
}

// Stars first .. first+count-1 of the table (0-based positions; star at position p is node p + 1).  r and phi
// are the table's arrays [n]; v_r, v_t and every output are the range's own arrays [count].
template <bool PAIRS>
__global__ void __launch_bounds__(ORB_THREADS, 1)
turning_points_kernel(uint32_t n, uint32_t first, uint32_t count, double G, const double* __restrict__ r, const double* __restrict__ v_r,
                      const double* __restrict__ v_t, const double* __restrict__ phi,
                      const Node* __restrict__ nodes, const double2* __restrict__ coarse_g,
                      const double2* __restrict__ mid_g, const uint32_t* __restrict__ dir, int shift, double* __restrict__ E_out, double* __restrict__ J_out, double* __restrict__ rmin_out,
                      double* __restrict__ rmax_out, uint32_t* __restrict__ kmin_out, uint32_t* __restrict__ kmax_out,
                      uint8_t* __restrict__ status_out, double* __restrict__ F_ws,
                      unsigned long long* __restrict__ counters)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* coarse = reinterpret_cast<double2*>(smem_raw);
    stage_coarse(coarse, coarse_g, n, shift);
    Tables T{ nodes, dir, coarse, shift > MID_SHIFT ? mid_g : nullptr, __ldg(r + (n - 1)), n, n >> shift, 1u << shift, shift, l2_keep_policy(), CoarseR{ reinterpret_cast<const double*>(coarse), 1 } };
    const uint32_t stride = gridDim.x * ORB_THREADS;
    const uint32_t lane = threadIdx.x & 31u;
    // whole warps stay in the loop together (the pair search is warp-collective); a lane beyond the end has no star
    for (uint32_t a = blockIdx.x * ORB_THREADS + threadIdx.x; PAIRS ? (a - lane < count) : (a < count); a += stride) {
        const bool valid = !PAIRS || a < count;
        const uint32_t b = valid ? a : count - 1;
        const Located L = locate_star(T, first + b, __ldcs(r + first + b), __ldcs(v_r + b), __ldcs(v_t + b), __ldcs(phi + first + b));
        const Solved v = PAIRS ? finish_star_s3_pairs(T, first + b, L, valid, lane) : finish_star_s3(T, first + b, L);
        if (!valid) continue;
        __stcs(F_ws + first + a, v.Fv);                            // by table position: a later S4 call may cover a sub-range
        __stcs(E_out + a, v.E); __stcs(J_out + a, v.J); __stcs(rmin_out + a, v.rmin); __stcs(rmax_out + a, v.rmax);
        __stcs(kmin_out + a, v.kmin); __stcs(kmax_out + a, v.kmax); status_out[a] = (uint8_t)v.st;
        if (v.st && counters) {
            if (v.st & HMC_STAR_UNBOUND) atomicAdd(counters + HMC_CNT_UNBOUND, 1ull);
            if (v.st & HMC_STAR_RADIAL) atomicAdd(counters + HMC_CNT_RADIAL, 1ull);
            if (v.st & HMC_STAR_DEGENERATE) atomicAdd(counters + HMC_CNT_DEGENERATE, 1ull);
        }
    }
}

// ---- S4 ---------------------------------------------------------------------------------------
struct Orbit {          // per-star constants of the draw
    double E, J, J2, mid, quarter, three_q, F;
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
    // X = ((w0 * 2^32 + w1) >> 11) * 2^-53 (R9).  The 53-bit integer is split into its top 21 and low 32
    // bits, converted separately (both exact) and added (exact: 53 bits): the same value as converting the
    // 64-bit integer, without the slow 64-bit integer-to-double conversion.
    const double X = u53_to_unit(w[0], w[1]);
    Trial tr;
    tr.Xp = u53_to_unit(w[2], w[3]);
    tr.s = 2.0 * X - 1.0;
    tr.r0 = o.mid + o.quarter * (3.0 * tr.s - (tr.s * tr.s) * tr.s);     // replaces Eq. 14 (R7)
    tr.w3 = w[3];
    return tr;
}

// coarse interval of r0, clamped to the orbit's own: largest c in [cl, ch] with coarse[c].r <= r0
__device__ __forceinline__ uint32_t coarse_locate(const CoarseR coarse, uint32_t cl, uint32_t ch, double r0)
{
    uint32_t lo = cl, hi = ch + 1;
    while (hi - lo > 1) {
        uint32_t m = (lo + hi) >> 1;
        if (coarse[m] <= r0) lo = m; else hi = m;
    }
    return lo;
}

// The same through an inverse table (S4 runs this once per trial: a quarter of its instructions were the twelve
// steps of the bisection above).  A radius is keyed by the leading bits of its binary64 pattern (exponent and top
// mantissa bits: monotone in r), INV_CELLS + 1 keys from that of r_1 on; inv[q] = largest coarse index whose
// radius is <= the smallest radius of key q.  The interval of r0 then lies in [inv[q], inv[q + 1]]: a handful of
// coarse entries instead of the orbit's few thousand.
#ifndef HMC_INV_CELLS_S4
#define HMC_INV_CELLS_S4 4096        // 2048: 0.705 ms, 4096: 0.699, 8192: 0.694 (and 2 us more set-up per launch), 16384: 0.750 at N = 1e7
#endif
static constexpr uint32_t INV_CELLS = 2048;            // fused kernel
static constexpr uint32_t INV_CELLS_S4 = HMC_INV_CELLS_S4;   // sampler proper

struct InvTable {
    const uint16_t* inv;     // shared memory, [INV_CELLS + 2]
    int base, sh;
    uint32_t cells;
    __device__ __forceinline__ uint32_t key(double x) const
    {
        const int q = (__double2hiint(x) >> sh) - base;
        return (uint32_t)min(max(q, 0), (int)cells - 1);
    }
};

// built by the whole CTA after stage_coarse; r_first, r_last: the radii of nodes 1 and N
__device__ __forceinline__ InvTable build_inv(uint16_t* inv, uint32_t cells, const CoarseR coarse, uint32_t ncoarse, double r_first, double r_last)
{
    InvTable t;
    t.cells = cells;
    const int h1 = __double2hiint(r_first), hn = __double2hiint(r_last);
    int sh = 0;
    while ((hn >> sh) - (h1 >> sh) > (int)cells - 1) ++sh;
    t.sh = sh; t.base = h1 >> sh; t.inv = inv;
    for (uint32_t q = threadIdx.x; q <= cells; q += ORB_THREADS) {
        const long long hw = ((long long)q + t.base) << sh;                   // leading word of the smallest radius of key q
        uint32_t lo = ncoarse;
        if (hw < 0x7ff00000ll) {
            const double x = __hiloint2double((int)hw, 0);
            lo = 0;
            uint32_t hi = ncoarse + 1;
            while (hi - lo > 1) { const uint32_t m = (lo + hi) >> 1; if (coarse[m] <= x) lo = m; else hi = m; }
        }
        // Key 0 also receives every radius BELOW r_1 (key() clamps from below), so its lower end must be coarse index 0
        // (r = 0), not the largest index <= r_1: where coarse[1] == r_1 and r_1 has zero low bits (a round innermost
        // radius with shift == 0, or 2^shift tied ones) that would be 1 and a trial inside the innermost star would be
        // given interval 1 instead of 0.
        inv[q] = (uint16_t)(q == 0 ? 0u : lo);
    }
    __syncthreads();
    return t;
}

__device__ __forceinline__ uint32_t coarse_locate(const CoarseR coarse, const InvTable& iv, uint32_t cl, uint32_t ch, double r0)
{
    const uint32_t q = iv.key(r0);
    uint32_t lo = iv.inv[q], hi = (uint32_t)iv.inv[q + 1] + 1;               // coarse[lo].r <= r0 < coarse[hi].r, or r0 < coarse[1].r
    while (hi - lo > 1) {
        const uint32_t m = (lo + hi) >> 1;
        if (coarse[m] <= r0) lo = m; else hi = m;
    }
    return min(max(lo, cl), ch);
}

// Exact evaluation of a trial, the oracle's expressions: shell j = #{ i : r_i <= r0 } clamped to
// [k_min, k_max], found from the directory of coarse interval c; Phi(r0) by Eq. 6 anchored at j; Q0; g.
__device__ __forceinline__ void exact_trial(const Tables& T, const Orbit& o, const Trial& tr, uint32_t c, double& Q0, double& g)
{
    uint32_t lo, hi;
    if (T.shift == 0) { lo = c; hi = c + 1; }          // the coarse table is the whole table
    else {
        T.dir_range(c, tr.r0, lo, hi);
        lo = max(lo, o.kmin); hi = min(hi, o.kmax + 1);
        if (hi <= lo) { lo = min(lo, o.kmax); hi = lo + 1; }
    }
    Node e = ld_node(T.nodes + lo);
    if (hi - lo > 1) {
        Node e1 = ld_node(T.nodes + lo + 1);
        if (e1.r <= tr.r0) {
            lo = lo + 1; e = e1;
            while (hi - lo > 1) {
                uint32_t p = (hi - lo > 4) ? lo + (hi - lo) / 2 : lo + 1;
                Node ep = ld_node(T.nodes + p);
                if (ep.r <= tr.r0) { lo = p; e = ep; } else hi = p;
            }
        }
    }
    const double phi0 = e.phi - e.B * (1.0 / tr.r0 - e.u);            // Eq. 6 anchored at node lo (R3)
    Q0 = 2.0 * (o.E - phi0) - o.J2 / (tr.r0 * tr.r0);                  // Eq. 12
    g = 0.0;
    if (Q0 > 0.0) g = (o.three_q * (1.0 - tr.s * tr.s)) / sqrt(Q0);
}

// Cold path, reached only if HMC_T_MAX trials were all rejected: redo the star exactly as the
// oracle's loop does, every trial evaluated, remembering the last trial with Q0 > 0.  Everything
// goes in and out by value so that nothing of the hot loop has its address taken (which would
// put it in local memory).
struct Exhaustive {
    double good_r, good_Q;
    uint32_t good_w3, used;
    unsigned st;
    bool accepted, have_good;
};

__device__ __noinline__ Exhaustive draw_exhaustive(Tables T, InvTable iv, Orbit o, uint32_t seed_lo, uint32_t seed_hi, uint32_t step,
                                                   unsigned st)
{
    Exhaustive x{ 0.0, 0.0, 0u, 0u, st, false, false };
    const uint32_t cl = o.kmin >> T.shift, ch = o.kmax >> T.shift;
    uint32_t t = 0;
    for (; t < HMC_T_MAX; ++t) {
        Trial tr = make_trial(o, seed_lo, seed_hi, step, t);
        double Q0, g;
        exact_trial(T, o, tr, coarse_locate(T.cr, iv, cl, ch, tr.r0), Q0, g);
        if (Q0 > 0.0) {
            x.have_good = true; x.good_r = tr.r0; x.good_Q = Q0; x.good_w3 = tr.w3;
            if (g > o.F) x.st |= HMC_STAR_CLIPPED;
            if (o.F * tr.Xp < g) { x.accepted = true; break; }
        }
    }
    x.used = x.accepted ? t + 1 : HMC_T_MAX;
    return x;
}

struct SampleIO {
    uint32_t first, count;   // the stars drawn are positions first .. first+count-1 of the table; per-star arrays are [count]
    const double *r, *v_r, *v_t, *E, *J, *rmin, *rmax;     // r: the table's radii [n]
    const uint32_t *kmin, *kmax, *id;
    const uint8_t* status_in;
    const double* F_ws;      // S3's bound F per star (workspace), or nullptr: compute it here
    const uint32_t* step_dev; // nullptr, or a device word added to the step number when the kernel runs (graph replay)
    uint32_t* batch_counter; // two workspace words, zero at launch (the table build zeroes them, this kernel's last CTA
                             // zeroes them again on its way out): [0] next unclaimed star, [1] CTAs that are done
    // fused S3 + S4 only: S3's table input and where its outputs go
    const double* phi;
    double *E_w, *J_w, *rmin_w, *rmax_w;
    uint32_t *kmin_w, *kmax_w;
    uint8_t* status_w;
    double *r_new, *v_r_new, *v_t_new;
    uint16_t* n_try;
    uint8_t* status_out;
    unsigned long long* counters;
};

// A warp's contiguous run of stars is written a few values at a time as the draws finish; plain
// (write-back) stores let L2 assemble whole sectors before they go to DRAM.
__device__ __forceinline__ void finish_star(const SampleIO& io, uint32_t a, double out_r, double out_vr, double out_vt,
                                            uint32_t used, unsigned st)
{
    io.r_new[a] = out_r; io.v_r_new[a] = out_vr; io.v_t_new[a] = out_vt;
    if (io.n_try) io.n_try[a] = (uint16_t)used;
    io.status_out[a] = (uint8_t)st;
    if (io.counters && (st & (HMC_STAR_CIRCULAR | HMC_STAR_MAXTRIES | HMC_STAR_CLIPPED))) {
        if (st & HMC_STAR_CIRCULAR) atomicAdd(io.counters + HMC_CNT_CIRCULAR, 1ull);
        if (st & HMC_STAR_MAXTRIES) atomicAdd(io.counters + HMC_CNT_MAXTRIES, 1ull);
        if (st & HMC_STAR_CLIPPED) atomicAdd(io.counters + HMC_CNT_CLIPPED, 1ull);
    }
}

// Per-warp parking area in shared memory: the orbits of the next (up to) 32 stars of the warp's
// run, prepared by all 32 lanes at once, from which lanes that have finished a star help
// themselves.  Preparing a batch costs one round of coalesced loads plus one round of node
// loads for the whole warp, instead of the same two round trips inside every trial iteration.
struct Park {
    double E[32], J[32], mid[32], delta[32], F[32];
    uint32_t kmin[32], kmax[32], sid[32], a[32], st[32];
};

// Prepare stars base .. base+31 (< end) from the S3 outputs.  Stars that take no draw (flagged by
// S3, or degenerate interval: CIRCULAR) are finished here.  Returns how many were parked.
__device__ __forceinline__ uint32_t park_from_arrays(const Node* __restrict__ nodes, const SampleIO& io, Park& pk,
                                                     uint32_t base, uint32_t end, uint32_t lane, unsigned lane_lt)
{
    const uint32_t a = base + lane;
    const bool in = a < end;
    unsigned st = 0;
    double E = 0.0, J = 0.0, rmin = 0.0, rmax = 0.0, F = 0.0;
    uint32_t kmin = 0, kmax = 0, sid = 0;
    if (in) {
        st = io.status_in[a];
        E = __ldcs(io.E + a); J = __ldcs(io.J + a);
        rmin = __ldcs(io.rmin + a); rmax = __ldcs(io.rmax + a);
        kmin = __ldcs(io.kmin + a); kmax = __ldcs(io.kmax + a);
        sid = __ldcs(io.id + a);
        if (io.F_ws) F = __ldcs(io.F_ws + io.first + a);
    }
    bool ok = in && !(st & (HMC_STAR_UNBOUND | HMC_STAR_RADIAL | HMC_STAR_DEGENERATE));
    const double delta = rmax - rmin;
    if (ok) {
        ok = delta > 0.0;
        if (ok && io.F_ws) ok = F > 0.0;
        else if (ok) {
            const double J2 = J * J;
            const double Bmin = ld_node(nodes + kmin).B, Bmax = ld_node(nodes + kmax).B;
            const double q1 = (2.0 * (J2 / rmin - Bmin)) / (rmin * rmin);      // Q'(r_min) in shell k_min
            const double q2 = (2.0 * (J2 / rmax - Bmax)) / (rmax * rmax);      // Q'(r_max) in shell k_max
            ok = (q1 > 0.0) && (q2 < 0.0);
            if (ok) F = 1.2 * fmax(sqrt((3.0 * delta) / q1), sqrt((3.0 * delta) / (-q2)));
        }
        if (!ok) st |= HMC_STAR_CIRCULAR;
    }
    if (in && !ok) finish_star(io, a, __ldg(io.r + io.first + a), __ldcs(io.v_r + a), __ldcs(io.v_t + a), 0u, st);
    const unsigned valid = __ballot_sync(0xffffffffu, ok);
    if (ok) {
        const uint32_t slot = __popc(valid & lane_lt);
        pk.E[slot] = E; pk.J[slot] = J; pk.mid[slot] = 0.5 * (rmin + rmax); pk.delta[slot] = delta; pk.F[slot] = F;
        pk.kmin[slot] = kmin; pk.kmax[slot] = kmax; pk.sid[slot] = sid; pk.a[slot] = a; pk.st[slot] = st;
    }
    __syncwarp();
    return (uint32_t)__popc(valid);
}

// Fused S3 + S4: prepare stars base .. base+31 by SOLVING them (S3's work, all 32 lanes busy), write S3's
// outputs, and park the orbits that take a draw; nothing of S3's output is read back.
__device__ __forceinline__ uint32_t park_by_solving(const Tables& T, const SampleIO& io, Park& pk, uint32_t base,
                                                    uint32_t end, uint32_t lane, unsigned lane_lt)
{
    const uint32_t a = base + lane;
    const bool in = a < end;
    bool ok = false;
    Solved v{ 0.0, 0.0, 0.0, 0.0, 0.0, 0u, 0u, 0u };
    uint32_t sid = 0;
    if (in) {
        const double rk = __ldcs(io.r + io.first + a), vr = __ldcs(io.v_r + a), vt = __ldcs(io.v_t + a), phik = __ldcs(io.phi + io.first + a);
        sid = __ldcs(io.id + a);
        v = solve_star(T, io.first + a, rk, vr, vt, phik);
        __stcs(io.E_w + a, v.E); __stcs(io.J_w + a, v.J); __stcs(io.rmin_w + a, v.rmin); __stcs(io.rmax_w + a, v.rmax);
        __stcs(io.kmin_w + a, v.kmin); __stcs(io.kmax_w + a, v.kmax); io.status_w[a] = (uint8_t)v.st;
        if (v.st && io.counters) {
            if (v.st & HMC_STAR_UNBOUND) atomicAdd(io.counters + HMC_CNT_UNBOUND, 1ull);
            if (v.st & HMC_STAR_RADIAL) atomicAdd(io.counters + HMC_CNT_RADIAL, 1ull);
            if (v.st & HMC_STAR_DEGENERATE) atomicAdd(io.counters + HMC_CNT_DEGENERATE, 1ull);
        }
        ok = !(v.st & (HMC_STAR_UNBOUND | HMC_STAR_RADIAL | HMC_STAR_DEGENERATE));
        if (ok) {
            ok = v.Fv > 0.0;                               // as S4 reading S3's F: 0 = empty interval or wrong end slopes
            if (!ok) v.st |= HMC_STAR_CIRCULAR;
        }
        if (!ok) finish_star(io, a, rk, vr, vt, 0u, v.st);
    }
    const unsigned valid = __ballot_sync(0xffffffffu, ok);
    if (ok) {
        const uint32_t slot = __popc(valid & lane_lt);
        pk.E[slot] = v.E; pk.J[slot] = v.J; pk.mid[slot] = 0.5 * (v.rmin + v.rmax); pk.delta[slot] = v.rmax - v.rmin; pk.F[slot] = v.Fv;
        pk.kmin[slot] = v.kmin; pk.kmax[slot] = v.kmax; pk.sid[slot] = sid; pk.a[slot] = a; pk.st[slot] = v.st;
    }
    __syncwarp();
    return (uint32_t)__popc(valid);
}

template <bool FUSED>
__device__ __forceinline__ void prefetch_inputs(const SampleIO& io, uint32_t a)
{
    if (FUSED) { prefetch_l2(io.r + io.first + a); prefetch_l2(io.v_r + a); prefetch_l2(io.v_t + a); prefetch_l2(io.phi + io.first + a); prefetch_l2(io.id + a); }
    else {
        prefetch_l2(io.E + a); prefetch_l2(io.J + a); prefetch_l2(io.rmin + a); prefetch_l2(io.rmax + a);
        prefetch_l2(io.kmin + a); prefetch_l2(io.kmax + a); prefetch_l2(io.id + a); prefetch_l2(io.status_in + a);
        if (io.F_ws) prefetch_l2(io.F_ws + io.first + a);
    }
}

template <bool FUSED>
__global__ void __launch_bounds__(ORB_THREADS, 1)
sample_new_radius_kernel(uint32_t n, double G, uint32_t seed_lo, uint32_t seed_hi, uint32_t step,
                         const Node* __restrict__ nodes, const double2* __restrict__ coarse_g,
                         const double2* __restrict__ mid_g, const uint32_t* __restrict__ dir, int shift, SampleIO io)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (io.step_dev) step += __ldg(io.step_dev);
    Park& pk = reinterpret_cast<Park*>(smem_raw)[threadIdx.x >> 5];
    // The coarse table.  Fused kernel: (r, Phi) pairs as in S3 (its search needs Phi exactly).  Sampler proper: the
    // radii as binary64 (they decide the coarse interval, hence the directory row, exactly) and Phi as binary32 beside
    // them: Phi is only used by the squeeze, whose bracket of Phi(r0) is a coarse interval wide (1e-4 relative) and is
    // simply widened by the binary32 rounding.  12 instead of 16 bytes per entry leave 39 KB more of the SM's 256 KB
    // to the L1 at N = 1e7, which this kernel's spills and streamed loads need: with a full table next to the
    // parking area nothing was left (sampling, ns per star: 0.0715 at N = 8e6, 0.0785 at 1.04e7, 0.0694 at 1.06e7).
    const uint32_t nc2 = (n >> shift) + 2;
    double2* coarse = nullptr;
    double* coarse_r = nullptr;
    float* coarse_phi = nullptr;
    unsigned char* after;
    if (FUSED) {
        coarse = reinterpret_cast<double2*>(smem_raw + ORB_WARPS * sizeof(Park));
        stage_coarse(coarse, coarse_g, n, shift);
        after = reinterpret_cast<unsigned char*>(coarse + nc2);
    } else {
        coarse_r = reinterpret_cast<double*>(smem_raw + ORB_WARPS * sizeof(Park));
        coarse_phi = reinterpret_cast<float*>(coarse_r + nc2);
        for (uint32_t c = threadIdx.x; c + 1 < nc2; c += ORB_THREADS) {
            const double2 e = __ldg(coarse_g + c);
            coarse_r[c] = e.x; coarse_phi[c] = (float)e.y;
        }
        if (threadIdx.x == 0) { coarse_r[nc2 - 1] = pos_inf(); coarse_phi[nc2 - 1] = 0.0f; }
        __syncthreads();
        after = reinterpret_cast<unsigned char*>(coarse_phi + ((nc2 + 1u) & ~1u));
    }
    const CoarseR cr = FUSED ? CoarseR{ reinterpret_cast<const double*>(coarse), 1 } : CoarseR{ coarse_r, 0 };
    Tables T{ nodes, dir, coarse, (FUSED && shift > MID_SHIFT) ? mid_g : nullptr, __ldg(io.r + (n - 1)), n, n >> shift, 1u << shift, shift, l2_keep_policy(), cr };
    const InvTable iv = build_inv(reinterpret_cast<uint16_t*>(after), FUSED ? INV_CELLS : INV_CELLS_S4, cr, T.ncoarse, __ldg(io.r), T.r_last);
    unsigned long long my_trials = 0;
    const unsigned lane_lt = lanemask_lt();
    const uint32_t lane = threadIdx.x & 31;

    // warps take batches of 32 consecutive stars from a global counter (the draws of some regions of the
    // cluster take longer than others: a static split leaves SMs idle at the end) and deal them to their lanes
    bool exhausted = false;
    uint32_t parked = 0, head = 0;          // park slots head .. parked-1 are waiting
    uint32_t next_base = 0;
    if (lane == 0) next_base = atomicAdd(io.batch_counter, 32u);
    next_base = __shfl_sync(0xffffffffu, next_base, 0);

    bool have = false;
    uint32_t a = 0, t = 0, cl = 0, ch = 0;
    unsigned st = 0;
    Orbit o;
    while (true) {
        // ---- deal parked orbits to the free lanes; prepare the next batch when the park runs dry
        unsigned need = __ballot_sync(0xffffffffu, !have);
        while (need) {
            if (head == parked) {
                if (exhausted) break;
                // the batch claimed one round ago is prepared now; the next one is claimed here and its
                // per-star inputs are pulled into L2 meanwhile
                const uint32_t base = next_base;
                if (base >= io.count) { exhausted = true; break; }
                if (lane == 0) next_base = atomicAdd(io.batch_counter, 32u);
                next_base = __shfl_sync(0xffffffffu, next_base, 0);
                if (next_base + lane < io.count) prefetch_inputs<FUSED>(io, next_base + lane);
                parked = FUSED ? park_by_solving(T, io, pk, base, io.count, lane, lane_lt)
                               : park_from_arrays(nodes, io, pk, base, io.count, lane, lane_lt);
                head = 0;
                continue;
            }
            const uint32_t slot = head + __popc(need & lane_lt);
            if (!have && slot < parked) {
                o.E = pk.E[slot]; o.J = pk.J[slot]; o.J2 = o.J * o.J; o.mid = pk.mid[slot];
                const double delta = pk.delta[slot];
                o.quarter = 0.25 * delta; o.three_q = 0.75 * delta; o.F = pk.F[slot];
                o.kmin = pk.kmin[slot]; o.kmax = pk.kmax[slot]; o.sid = pk.sid[slot];
                a = pk.a[slot]; st = pk.st[slot];
                cl = o.kmin >> shift; ch = o.kmax >> shift;
                t = 0;
                have = true;
            }
            head = min(parked, head + (uint32_t)__popc(need));
            __syncwarp();
            need = __ballot_sync(0xffffffffu, !have);
        }
        if (!__any_sync(0xffffffffu, have)) break;          // nothing parked, nothing left to prepare
        // ---- up to FRONT_ROUNDS trials for every lane that holds a star, until one survives the squeeze.
        // Half the trials are rejected by the squeeze alone; a lane whose trial was, tries its next one at
        // once instead of idling through the other lanes' exact look-ups (which cost more than a trial's front
        // part), so fewer of the expensive rounds are needed per star.
        bool candidate = false;
        Trial tr{ 0.0, 0.0, 0.0, 0u };
        uint32_t c = 0;
#pragma unroll 1
        for (int round = 0; round < FRONT_ROUNDS; ++round) {
            if (have && !candidate && t < HMC_T_MAX) {
                tr = make_trial(o, seed_lo, seed_hi, step, t);
                c = coarse_locate(cr, iv, cl, ch, tr.r0);
                ++t;
                // squeeze: Phi(r0) lies in [coarse[c].Phi, coarse[c+1].Phi]; everything widened by ~1e-11.
                // Written multiplied through by r0^2 > 0, so there is no division on this path.
                const double r2 = tr.r0 * tr.r0;
                double phi_lo, phi_hi;                                      // Phi_c <= Phi(r0) <= Phi_{c+1}, bounded from outside
                if (FUSED) { phi_lo = coarse[c].y; phi_hi = coarse[c + 1].y; }
                else {      // binary32 copies: off by at most 2^-24 relative (or 2^-150 absolute); widened by twice that
                    const double a = (double)coarse_phi[c], b = (double)coarse_phi[c + 1];
                    phi_lo = a - (1.25e-7 * fabs(a) + 3e-45);
                    phi_hi = b + (1.25e-7 * fabs(b) + 3e-45);
                }
                const double top = 2.0 * (o.E - phi_lo) * r2;
                const double tol = 1e-11 * (fabs(top) + o.J2);
                const double Qh = (top - o.J2) + tol;                       // upper bound of r0^2 Q0
                candidate = !(Qh <= 0.0);                                   // (a NaN from overflowing bounds keeps the trial)
                if (candidate) {
                    const double Ql = (2.0 * (o.E - phi_hi) * r2 - o.J2) - tol;   // lower bound of r0^2 Q0
                    const double fx = o.F * tr.Xp, cc = o.three_q * (1.0 - tr.s * tr.s);
                    if (Ql > 0.0 && (fx * fx) * Ql > ((cc * cc) * r2) * (1.0 + 1e-10)) candidate = false;   // F X' > g for certain
                }
            }
            if (__all_sync(0xffffffffu, !have || candidate || t >= HMC_T_MAX)) break;
        }
        if (have) {
            bool done = false, accepted = false, have_good = false;
            double good_r = 0.0, good_Q = 0.0;
            uint32_t good_w3 = 0, used = t;
            if (candidate) {
                double Q0, g;
                exact_trial(T, o, tr, c, Q0, g);
                if (Q0 > 0.0) {
                    if (g > o.F) st |= HMC_STAR_CLIPPED;
                    if (o.F * tr.Xp < g) { done = accepted = have_good = true; good_r = tr.r0; good_Q = Q0; good_w3 = tr.w3; }
                }
            }
            if (!done && t >= HMC_T_MAX) {
                const Exhaustive x = draw_exhaustive(T, iv, o, seed_lo, seed_hi, step, st);
                st = x.st; accepted = x.accepted; used = x.used; have_good = x.have_good;
                good_r = x.good_r; good_Q = x.good_Q; good_w3 = x.good_w3;
                done = true;
            }
            if (done) {
                my_trials += used;
                if (!accepted) st |= HMC_STAR_MAXTRIES;
                double out_r, out_vr, out_vt;
                if (have_good) {
                    out_r = good_r;
                    out_vt = o.J / good_r;
                    const double vrn = sqrt(good_Q);                    // v_r = Q^(1/2)
                    out_vr = (good_w3 & 1u) ? -vrn : vrn;
                } else { out_r = __ldg(io.r + io.first + a); out_vr = __ldcs(io.v_r + a); out_vt = __ldcs(io.v_t + a); }
                finish_star(io, a, out_r, out_vr, out_vt, used, st);
                have = false;
            }
        }
    }
    if (io.counters) {
        for (int off = 16; off > 0; off >>= 1) my_trials += __shfl_down_sync(0xffffffffu, my_trials, off);
        if ((threadIdx.x & 31) == 0 && my_trials) atomicAdd(io.counters + HMC_CNT_TRIALS, my_trials);
    }
    // leave the two counter words as they were found, for a next S4 launch on the same tables (ranges of one table)
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(io.batch_counter + 1, 1u) == gridDim.x - 1) { io.batch_counter[0] = 0; io.batch_counter[1] = 0; __threadfence(); }
    }
}

// ---- energy correction for the time-varying potential (R18) ------------------
// Per star, in the NEW sorted order: Phi'(r_old) from the new table (coarse interval by bisection in
// shared memory, node by the directory, Eq. 6 anchored at the node), then the oracle's expressions.
__global__ void __launch_bounds__(ORB_THREADS, 1)
energy_correction_kernel(uint32_t n, const Node* __restrict__ nodes, const double2* __restrict__ coarse_g,
                         const uint32_t* __restrict__ dir, int shift, const double* __restrict__ r,
                         const double* __restrict__ phi, const double* __restrict__ E_old,
                         const double* __restrict__ r_old, const double* __restrict__ p_old,
                         const double* __restrict__ v_r, const double* __restrict__ v_t, double* __restrict__ v_r_out,
                         double* __restrict__ v_t_out, uint8_t* __restrict__ status_out,
                         unsigned long long* __restrict__ counters)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* coarse = reinterpret_cast<double2*>(smem_raw);
    stage_coarse(coarse, coarse_g, n, shift);
    Tables T{ nodes, dir, coarse, nullptr, __ldg(r + (n - 1)), n, n >> shift, 1u << shift, shift, l2_keep_policy(), CoarseR{ reinterpret_cast<const double*>(coarse), 1 } };
    const uint32_t stride = gridDim.x * ORB_THREADS;
    for (uint32_t a = blockIdx.x * ORB_THREADS + threadIdx.x; a < n; a += stride) {
        const double x = __ldcs(r_old + a);
        double vr = __ldcs(v_r + a), vt = __ldcs(v_t + a);
        const double E = __ldcs(E_old + a), po = __ldcs(p_old + a), ph = __ldcs(phi + a);
        // shell of r_old in the new table: j = #{ i : r_i <= x }, 0 .. n
        const uint32_t c = coarse_locate(T.cr, 0u, T.ncoarse, x);
        uint32_t lo, hi;
        if (shift == 0) { lo = c; hi = c + 1; }
        else T.dir_range(c, x, lo, hi);
        Node e = ld_node(nodes + lo);
        while (hi - lo > 1) {
            const uint32_t p = (hi - lo > 4) ? lo + (hi - lo) / 2 : lo + 1;
            const Node ep = ld_node(nodes + p);
            if (ep.r <= x) { lo = p; e = ep; } else hi = p;
        }
        const double po2 = e.phi - e.B * (1.0 / x - e.u);                  // Phi'(r_old), Eq. 6 anchored (R3)
        const double K = 0.5 * (vr * vr + vt * vt);
        const double pn = E - K;                                           // Phi(r_new): the draw's energy identity
        const double dE = 0.5 * ((po2 - po) + (ph - pn));
        const double Kp = (E + dE) - ph;
        unsigned st = 0;
        if (Kp > 0.0 && K > 0.0) {
            const double lam = sqrt(Kp / K);
            vr = lam * vr; vt = lam * vt;
        } else st |= HMC_STAR_NOKINETIC;
        __stcs(v_r_out + a, vr); __stcs(v_t_out + a, vt); status_out[a] = (uint8_t)st;
        if (st && counters) atomicAdd(counters + HMC_CNT_NOKINETIC, 1ull);
    }
}

// ---- host side --------------------------------------------------------------------------------
// S3's exact search by lane pairs pays when the node table is far beyond the TLB's reach (see probe_pairs).
// Turning-point stage, one lane / lane pairs, ms: N = 1e7 0.90 / 1.40, 3.4e7 5.1 / 5.0, 4.2e7 6.9 / 6.3, 5e7 8.8 / 7.6,
// 1e8 20.6 / 16.0.
// (A test-only build sets the threshold to 1 so that small cases run the pair search: build.py "pairs".)
#ifndef HMC_S3_PAIRS_MIN_N
#define HMC_S3_PAIRS_MIN_N (1ull << 25)
#endif
static inline bool s3_pairs(uint64_t n) { return n >= HMC_S3_PAIRS_MIN_N; }

static hmc_status build_tables(uint64_t n, double G, const double* r, const double* phi, const double* m_cum,
                               const Workspace& ws, int shift, cudaStream_t st)
{
    if (shift == 0) {                                            // the coarse table is the whole table: no directory
        const int blocks = (int)umin64((n + 2 + 255) / 256, (uint64_t)sm_count() * 8);
        build_nodes_kernel<<<blocks, 256, 0, st>>>(r, phi, m_cum, G, ws.nodes, ws.coarse, ws.mid, shift, n, ws.tickets + 16);
        HMC_LAUNCH_CHECK();
        return HMC_OK;
    }
    if ((1 << shift) <= DIR_SMALL_MAX_K) {                        // shift <= MID_SHIFT here: no mid table
        const uint32_t nintervals = (uint32_t)((n >> shift) + 1);
        build_tables_small_kernel<<<(nintervals + DIR_THREADS / 32 - 1) / (DIR_THREADS / 32), DIR_THREADS, 0, st>>>(
            r, phi, m_cum, G, ws.nodes, ws.coarse, ws.dir, (uint32_t)n, shift, nintervals, ws.tickets + 16);
        HMC_LAUNCH_CHECK();
        return HMC_OK;
    }
    const size_t smem = ((size_t)(1u << shift) + 1) * sizeof(uint32_t);
    static std::atomic<uint64_t> opted{ 0 };                      // the largest row any n <= HMC_MAX_N needs
    hmc_status so = smem_opt_in(opted, build_tables_kernel, ((size_t)(1u << coarse_shift(HMC_MAX_N)) + 1) * sizeof(uint32_t));
    if (so != HMC_OK) return so;
    build_tables_kernel<<<(unsigned)((n >> shift) + 1), DIR_THREADS, smem, st>>>(r, phi, m_cum, G, ws.nodes, ws.coarse, ws.mid,
                                                                                 ws.dir, (uint32_t)n, shift, ws.tickets + 16);
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

hmc_status turning_points(uint64_t n, uint64_t first, uint64_t count, double G, const double* r, const double* v_r, const double* v_t,
                          const double* phi, const double* m_cum, double* E, double* J, double* r_min,
                          double* r_max, uint32_t* k_min, uint32_t* k_max, uint8_t* status, uint64_t* counters,
                          const Workspace& ws, cudaStream_t st, bool reuse_tables)
{
    const int sms = sm_count();
    const int shift = coarse_shift(n);
    const bool pairs = s3_pairs(n);
    const size_t smem = ((n >> shift) + 2) * sizeof(double2);
    static std::atomic<uint64_t> opted[2];
    hmc_status so = pairs ? smem_opt_in(opted[1], turning_points_kernel<true>, COARSE_CAP * sizeof(double2))
                          : smem_opt_in(opted[0], turning_points_kernel<false>, COARSE_CAP * sizeof(double2));
    if (so != HMC_OK) return so;
    hmc_status s = reuse_tables ? HMC_OK : build_tables(n, G, r, phi, m_cum, ws, shift, st);
    if (s != HMC_OK) return s;
    if (count == 0) return HMC_OK;
    const int blocks = (int)umin64((count + ORB_THREADS - 1) / ORB_THREADS, (uint64_t)sms);
    if (pairs)
        turning_points_kernel<true><<<blocks, ORB_THREADS, smem, st>>>((uint32_t)n, (uint32_t)first, (uint32_t)count, G, r, v_r, v_t, phi, ws.nodes, ws.coarse, ws.mid, ws.dir, shift,
                                                                      E, J, r_min, r_max, k_min, k_max, status, ws.orbitF,
                                                                      reinterpret_cast<unsigned long long*>(counters));
    else
        turning_points_kernel<false><<<blocks, ORB_THREADS, smem, st>>>((uint32_t)n, (uint32_t)first, (uint32_t)count, G, r, v_r, v_t, phi, ws.nodes, ws.coarse, ws.mid, ws.dir, shift,
                                                                       E, J, r_min, r_max, k_min, k_max, status, ws.orbitF,
                                                                       reinterpret_cast<unsigned long long*>(counters));
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

static hmc_status launch_sampler(bool fused, uint64_t n, double G, uint64_t seed, uint32_t step, int shift, const SampleIO& io_in,
                                 const Workspace& ws, cudaStream_t st)
{
    const int sms = sm_count();
    const size_t inv_bytes = ((fused ? INV_CELLS : INV_CELLS_S4) + 2) * sizeof(uint16_t);
    // fused: (r, Phi) pairs; sampler proper: radii as binary64 + Phi as binary32 (an even number of them)
    const size_t nc2 = (n >> shift) + 2;
    const size_t smem = ORB_WARPS * sizeof(Park) + (fused ? nc2 * sizeof(double2) : nc2 * sizeof(double) + ((nc2 + 1) & ~(size_t)1) * sizeof(float)) + inv_bytes;
    static std::atomic<uint64_t> opted[2];
    const size_t cap = ORB_WARPS * sizeof(Park) + COARSE_CAP * (fused ? sizeof(double2) : sizeof(double) + sizeof(float)) + inv_bytes;
    hmc_status so = fused ? smem_opt_in(opted[1], sample_new_radius_kernel<true>, cap)
                          : smem_opt_in(opted[0], sample_new_radius_kernel<false>, cap);
    if (so != HMC_OK) return so;
    if (io_in.count == 0) return HMC_OK;
    const int blocks = (int)umin64(((uint64_t)io_in.count + ORB_THREADS - 1) / ORB_THREADS, (uint64_t)sms);
    SampleIO io = io_in;
    io.batch_counter = ws.tickets + 16;
    if (fused)
        sample_new_radius_kernel<true><<<blocks, ORB_THREADS, smem, st>>>((uint32_t)n, G, (uint32_t)seed, (uint32_t)(seed >> 32), step,
                                                                         ws.nodes, ws.coarse, ws.mid, ws.dir, shift, io);
    else
        sample_new_radius_kernel<false><<<blocks, ORB_THREADS, smem, st>>>((uint32_t)n, G, (uint32_t)seed, (uint32_t)(seed >> 32), step,
                                                                          ws.nodes, ws.coarse, ws.mid, ws.dir, shift, io);
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

hmc_status sample_new_radius(uint64_t n, uint64_t first, uint64_t count, double G, uint64_t seed, uint32_t step, const double* r,
                             const double* phi, const double* m_cum, const double* v_r, const double* v_t,
                             const double* E, const double* J, const double* r_min, const double* r_max,
                             const uint32_t* k_min, const uint32_t* k_max, const uint32_t* id,
                             const uint8_t* status_in, double* r_new, double* v_r_new, double* v_t_new,
                             uint16_t* n_try, uint8_t* status_out, uint64_t* counters, bool reuse_tables,
                             const Workspace& ws, cudaStream_t st, const uint32_t* step_dev)
{
    const int shift = coarse_shift(n);
    if (!reuse_tables) {
        hmc_status s = build_tables(n, G, r, phi, m_cum, ws, shift, st);
        if (s != HMC_OK) return s;
    }
    SampleIO io{};
    io.first = (uint32_t)first; io.count = (uint32_t)count;
    io.r = r; io.v_r = v_r; io.v_t = v_t; io.E = E; io.J = J; io.rmin = r_min; io.rmax = r_max;
    io.kmin = k_min; io.kmax = k_max; io.id = id; io.status_in = status_in;
    io.F_ws = reuse_tables ? ws.orbitF : nullptr;
    io.step_dev = step_dev;
    io.r_new = r_new; io.v_r_new = v_r_new; io.v_t_new = v_t_new; io.n_try = n_try; io.status_out = status_out;
    io.counters = reinterpret_cast<unsigned long long*>(counters);
    return launch_sampler(false, n, G, seed, step, shift, io, ws, st);
}

hmc_status energy_correction(uint64_t n, double G, const double* r, const double* phi, const double* m_cum,
                             const double* E_old, const double* r_old, const double* p_old, const double* v_r,
                             const double* v_t, double* v_r_out, double* v_t_out, uint8_t* status_out,
                             uint64_t* counters, const Workspace& ws, cudaStream_t st)
{
    const int sms = sm_count();
    const int shift = coarse_shift(n);
    const size_t smem = ((n >> shift) + 2) * sizeof(double2);
    static std::atomic<uint64_t> opted{ 0 };
    hmc_status so = smem_opt_in(opted, energy_correction_kernel, COARSE_CAP * sizeof(double2));
    if (so != HMC_OK) return so;
    hmc_status s = build_tables(n, G, r, phi, m_cum, ws, shift, st);
    if (s != HMC_OK) return s;
    const int blocks = (int)umin64((n + ORB_THREADS - 1) / ORB_THREADS, (uint64_t)sms);
    energy_correction_kernel<<<blocks, ORB_THREADS, smem, st>>>((uint32_t)n, ws.nodes, ws.coarse, ws.dir, shift, r, phi, E_old,
                                                               r_old, p_old, v_r, v_t, v_r_out, v_t_out, status_out,
                                                               reinterpret_cast<unsigned long long*>(counters));
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

__global__ void add_u32_kernel(uint32_t* p, uint32_t inc) { *p += inc; }

hmc_status add_u32(uint32_t* p, uint32_t inc, cudaStream_t st)
{
    add_u32_kernel<<<1, 1, 0, st>>>(p, inc);
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

// the tables alone (what every S3 call and an S4 call without reuse_tables start with)
hmc_status orbit_build_tables(uint64_t n, double G, const double* r, const double* phi, const double* m_cum, const Workspace& ws,
                              cudaStream_t st)
{
    return build_tables(n, G, r, phi, m_cum, ws, coarse_shift(n), st);
}

// S3 + S4 in one launch: same outputs as the two calls.
hmc_status orbit_step(uint64_t n, uint64_t first, uint64_t count, double G, uint64_t seed, uint32_t step, const double* r, const double* v_r,
                      const double* v_t, const double* phi, const double* m_cum, const uint32_t* id, double* E,
                      double* J, double* r_min, double* r_max, uint32_t* k_min, uint32_t* k_max, uint8_t* status,
                      double* r_new, double* v_r_new, double* v_t_new, uint16_t* n_try, uint8_t* status_out,
                      uint64_t* counters, const Workspace& ws, cudaStream_t st)
{
    const int shift = coarse_shift(n);
    hmc_status s = build_tables(n, G, r, phi, m_cum, ws, shift, st);
    if (s != HMC_OK) return s;
    SampleIO io{};
    io.first = (uint32_t)first; io.count = (uint32_t)count;
    io.r = r; io.v_r = v_r; io.v_t = v_t; io.id = id; io.phi = phi;
    io.E_w = E; io.J_w = J; io.rmin_w = r_min; io.rmax_w = r_max; io.kmin_w = k_min; io.kmax_w = k_max; io.status_w = status;
    io.r_new = r_new; io.v_r_new = v_r_new; io.v_t_new = v_t_new; io.n_try = n_try; io.status_out = status_out;
    io.counters = reinterpret_cast<unsigned long long*>(counters);
    return launch_sampler(true, n, G, seed, step, shift, io, ws, st);
}

}  // namespace hmc
