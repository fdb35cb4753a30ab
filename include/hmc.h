/*
 * hmc.h -- C ABI of libhmc: the per-timestep orbit computation of the Henon Monte Carlo
 * method (arXiv 1206.5878, Pattabiraman et al.; cited as PAPER.md:LINE) on one NVIDIA B200.
 *
 * One "orbit step" over N spherically symmetric stars is four calls, in this order:
 *
 *   hmc_sort_by_radius        PAPER.md:139  (step 6, "Sort stars by radial distance")
 *   hmc_potential             PAPER.md:67-79 (step 1, Eq. 1-5)
 *   hmc_orbit_turning_points  PAPER.md:117-124 (step 5, Eq. 12, bracket + analytic roots)
 *   hmc_sample_new_radius     PAPER.md:126-137 (step 5, Eq. 13-15, rejection sampling)
 * (hmc_orbit_step does the last two in one launch.)
 *
 * Conventions common to all calls
 * -------------------------------
 *  - Unless a parameter says "host", every array pointer is a DEVICE pointer owned by the
 *    caller.  The library never allocates, frees or keeps device memory between calls; scratch
 *    space is the caller's `workspace` of at least hmc_workspace_bytes(n) bytes, 256-byte aligned.
 *    (The one thing it keeps: hmc_step_host's two streams and their events, see there; and a launch counter.
 *    hmc_potential_static takes no workspace: its scratch is a fixed array inside the library image, see there.)
 *  - Every call is asynchronous on `cuda_stream` (a cudaStream_t passed as void*; NULL = the
 *    legacy default stream) and never synchronises the host.
 *  - Inputs are never modified; outputs must not alias inputs or each other.
 *  - fp64 arrays must be 8-byte aligned, uint32 arrays 4-byte aligned.
 *  - Arrays are 0-based; element a of a radius-sorted array is the paper's star k = a + 1.
 *    Shell indices k_min / k_max use the paper's numbering: shell j is [r_j, r_{j+1}],
 *    j = 0 (inside the innermost star) ... N (beyond the outermost star).
 *  - n == 0 is a no-op returning HMC_OK.  n > HMC_MAX_N returns HMC_ERR_SIZE.
 *  - Return value: HMC_OK or a negative call-level error; nothing is thrown.  A launch failure
 *    returns HMC_ERR_CUDA and leaves the CUDA error readable through cudaGetLastError().
 *  - Per-star data problems never fail a call: they set bits in `star_status` and the star is
 *    left where it is (r_new = r, velocities unchanged).
 *  - Arithmetic is IEEE-754 binary64 throughout, without fused multiply-add contraction; the
 *    operation order of every formula is fixed in DESIGN.md ("Readings", R1p-R9) so that results
 *    can be compared bit for bit with a CPU evaluation of the same formulas.
 *  - Thread safety: calls are re-entrant when they use distinct workspaces.
 */
#ifndef HMC_H
#define HMC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef int32_t hmc_status;

#if defined(__GNUC__)
#define HMC_API __attribute__((visibility("default")))
#else
#define HMC_API
#endif

#define HMC_OK              0
#define HMC_ERR_NULL       (-1)  /* a required pointer is NULL                              */
#define HMC_ERR_SIZE       (-2)  /* n > HMC_MAX_N, or ncols out of range                    */
#define HMC_ERR_WORKSPACE  (-3)  /* workspace NULL, misaligned or smaller than required     */
#define HMC_ERR_ALIGN      (-4)  /* an array pointer is not aligned to its element size     */
#define HMC_ERR_CUDA       (-5)  /* a CUDA runtime call or kernel launch failed             */

#define HMC_MAX_N      (1ull << 28)   /* stars per call                                     */
#define HMC_MAX_COLS   8              /* fp64 record columns carried by the sort            */
#define HMC_MAX_PEERS  16             /* further copies of the table hmc_potential_shard_push writes to */

/* star_status bits */
#define HMC_STAR_UNBOUND     1u   /* E >= 0 (or NaN): no apocentre; r_max = +inf, no draw           */
#define HMC_STAR_RADIAL      2u   /* J^2 == 0: pericentre at r = 0; no draw                         */
#define HMC_STAR_DEGENERATE  4u   /* outer quadratic has C >= 0 (cannot happen for a genuine bracket)*/
#define HMC_STAR_CIRCULAR    8u   /* r_max - r_min <= 0 or end slopes of the wrong sign; no draw    */
#define HMC_STAR_MAXTRIES   16u   /* rejection loop reached HMC_T_MAX trials                        */
#define HMC_STAR_CLIPPED    32u   /* some trial had g > F (density clipped there); draw still valid */
#define HMC_STAR_NOKINETIC  64u   /* energy correction: corrected kinetic energy <= 0; velocities kept */

#ifndef HMC_T_MAX                 /* (a test-only build lowers it to reach the exhaustion path) */
#define HMC_T_MAX   4096u         /* cap on rejection trials per star (R7)        */
#endif

/* device counters accumulated (atomically) by the orbit calls; the caller zeroes them */
enum {
    HMC_CNT_UNBOUND = 0, HMC_CNT_RADIAL, HMC_CNT_DEGENERATE, HMC_CNT_CIRCULAR,
    HMC_CNT_MAXTRIES, HMC_CNT_CLIPPED, HMC_CNT_TRIALS, HMC_CNT_NOKINETIC,
    HMC_NCOUNTERS
};

/* Bytes of scratch any of the calls below may need for n stars (the maximum over the calls; about
 * 132 bytes per star: the sort's packed words and 64-byte star records, the 32-byte search nodes of the
 * orbit calls, their radius directory, and S3's per-star bound for S4). */
HMC_API size_t hmc_workspace_bytes(uint64_t n);

/* Static string for a status code. */
HMC_API const char* hmc_status_string(hmc_status s);

/* Library version as major*10000 + minor*100 + patch. */
HMC_API int32_t hmc_version(void);

/* The cap on rejection trials this build was compiled with (HMC_T_MAX). */
HMC_API uint32_t hmc_t_max(void);

/* Number of CUDA kernels this process has launched through the library so far (all threads, all devices;
 * memsets and copies are not kernels).  A monotone counter for accounting: bench.py reports the difference
 * over its timed region as `gpu_launches`. */
HMC_API uint64_t hmc_launch_count(void);

/*
 * S1  "Sort stars by radial distance".
 * Produces the unique ascending order by the pair (r_i, i): a stable sort, ties kept in
 * input order (the paper's Quicksort leaves tie order open; R1).
 *   r_in[n]        radii, finite and > 0 (their bit patterns are sorted as unsigned integers)
 *   r_sorted[n]    out: radii ascending
 *   perm[n]        out: perm[k] = index into r_in of the k-th smallest radius
 *   ncols          0..HMC_MAX_COLS record columns to carry along
 *   cols_in/out    HOST arrays of ncols DEVICE pointers: cols_out[c][k] = cols_in[c][perm[k]]
 *   id_in/id_out   optional (both or neither NULL) persistent star-id column, gathered likewise
 * Method: each star is one 64-bit word (leading key bits above the smallest key | index); a stable
 * least-significant-digit radix sort of those words (8-bit digits, one decoupled-look-back sweep
 * per digit), then one kernel that resolves runs of stars agreeing in the kept key bits from
 * their full keys and moves the record columns (as one 64-byte record per star when ncols <= 6).
 * A run of more than 32 such stars makes the general sort (eight passes over 64-bit key +
 * 32-bit index, enqueued behind a device-side flag) redo the call.  The result is the same
 * unique permutation either way.
 */
HMC_API hmc_status hmc_sort_by_radius(uint64_t n,
        const double* r_in, double* r_sorted, uint32_t* perm,
        int32_t ncols, const double* const* cols_in, double* const* cols_out,
        const uint32_t* id_in, uint32_t* id_out,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * S2  "Potential calculation".  On radius-sorted r, m:
 *   m_cum[k] = M_k   = sum_{i<=k} m_i                       (Eq. 3, 5)
 *   phi[k]   = Phi_k = -G ( M_k / r_k + sum_{i>k} m_i / r_i )   (Eq. 1 at r = r_k; == Eq. 2-5)
 * Both sums are accumulated in double-double and rounded once (R1p).
 * Preconditions: r ascending, finite, > 0; m >= 0.
 */
HMC_API hmc_status hmc_potential(uint64_t n, double G,
        const double* r_sorted, const double* m_sorted,
        double* phi, double* m_cum,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * S2 for callers that cannot allocate device memory: hmc_potential without a workspace argument.
 *
 * Who this is for.  Every other call here needs a `workspace` the caller obtained from cudaMalloc (or from a pool
 * that did).  Some callers cannot do that at the point where they need Phi: code running inside a host program
 * whose device memory is handed out once at start-up by an allocator the plug-in may not call (a simulation
 * framework's arena, a job with a fixed memory budget that fails if the driver allocates behind its back), a
 * callback that runs while another thread holds the allocator's lock, or a real-time loop in which cudaMalloc's
 * implicit device synchronisation is not acceptable.  Such a caller already owns r, m, phi and m_cum (its own
 * star arrays); what it lacks is the few hundred kilobytes of partial sums the two launches of S2 hand to each
 * other.  This entry point keeps those in an array that is part of the library image itself.
 *
 * What it computes: exactly hmc_potential (Eq. 1-5; same two kernels, same launch
 * configuration, same bits): m_cum[k] = M_k, phi[k] = -G (M_k / r_k + sum_{i>k} m_i / r_i).
 *
 * The scratch: a file-scope `static __device__` array in hmc_potential.cu of HMC_STATIC_SCRATCH_BYTES bytes
 * (544 KiB), 256-byte aligned.  Every GPU on which this process uses the library holds one copy from the moment
 * the library's device code is loaded there until the process exits, whether or not this call is ever made.
 * It holds one 32-byte total per 1024 stars plus one per CTA of the launch, hence the limit
 *     n <= HMC_STATIC_MAX_N = 2^24 (16 777 216 stars);
 * a larger n returns HMC_ERR_STATIC_LIMIT and launches nothing (use hmc_potential with a workspace instead).
 * The same status is returned on a GPU with more than 341 multiprocessors (more CTAs than the array has room for).
 *
 * Set-up: the first call on each device looks up the array's device address (cudaGetSymbolAddress, with that
 * device current) and remembers it for the process.  That look-up may make the CUDA runtime load the library's
 * device code, so make the first call on a device OUTSIDE any stream capture; later calls only launch kernels.
 * The call itself never calls cudaMalloc, cudaFree or any routine that allocates, on the host or the device.
 *
 * Sharing: there is ONE array per device, used by every call from every thread and stream.  Nothing in it has
 * to start at zero (the first launch overwrites every entry the second one reads, so the previous call's
 * contents do no harm), but two calls whose kernels may run at the same time on one device -- different
 * streams, or different host threads on different streams -- overwrite each other's partial sums and produce
 * wrong potentials without any error.  Calls on one stream, or ordered by events, are safe.
 * Everything else (argument rules, asynchrony, n == 0) is as for hmc_potential.
 */
#define HMC_STATIC_MAX_N          (1ull << 24)
#define HMC_STATIC_SCRATCH_BYTES  ((16384u + 1024u) * 32u)
#define HMC_ERR_STATIC_LIMIT      (-6)  /* n (or the GPU's SM count) beyond what the built-in scratch array holds */

HMC_API hmc_status hmc_potential_static(uint64_t n, double G,
        const double* r_sorted, const double* m_sorted,
        double* phi, double* m_cum, void* cuda_stream);

/*
 * S3  Pericentre and apocentre of every star's orbit.
 * For star k:  E = Phi_k + (v_r^2 + v_t^2)/2  (Eq. 16),  J = r_k v_t,
 *   Q(r) = 2E - 2Phi(r) - J^2/r^2  (Eq. 12);
 *   k_min = largest  j <= k-1 with Q(r_j) < 0   (node 0, r = 0, counts as negative)
 *   k_max = (smallest j >= k+1 with Q(r_j) < 0) - 1   (node N+1, r = inf, counts as negative)
 *   r_min / r_max = root of Q inside shell k_min / k_max, where Phi = Phi_j - G M_j (1/r - 1/r_j)
 *   makes Q quadratic in 1/r (closed form; R3, R5).
 * Outputs are [n] in the same (sorted) order.  star_status gets UNBOUND / RADIAL / DEGENERATE.
 * counters: device uint64[HMC_NCOUNTERS], accumulated; may be NULL.
 */
HMC_API hmc_status hmc_orbit_turning_points(uint64_t n, double G,
        const double* r_sorted, const double* v_r, const double* v_t,
        const double* phi, const double* m_cum,
        double* E, double* J, double* r_min, double* r_max,
        uint32_t* k_min, uint32_t* k_max, uint8_t* star_status,
        uint64_t* counters,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * S4  New radial position on the orbit: von Neumann rejection with density
 * proportional to 1/|v_r|, v_r = sqrt(Q(r)) (Eq. 13-15), in the variable s of DESIGN.md R7 that
 * removes the end-point singularities the paper mentions.
 * Trial t of the star with persistent id `id[k]` at step `step` uses
 * Philox4x32-10(counter = (id, 0, step, t), key = (seed low word, seed high word)); a star's
 * draw therefore does not depend on its position in the arrays (R9).
 *   tables   r_sorted, phi, m_cum [n]
 *   per star E, J, r_min, r_max, k_min, k_max, star_status_in (outputs of S3), id,
 *            v_r, v_t (copied through for stars that are not drawn)
 *   outputs  r_new, v_r_new, v_t_new [n]; n_try[n] (trials used, may be NULL);
 *            star_status_out[n] (input bits plus CIRCULAR / MAXTRIES / CLIPPED)
 * v_t_new = J / r_new, v_r_new = +-sqrt(Q(r_new)) with the sign from a spare random bit.
 *   reuse_tables  S3 and S4 search the same tables, which each call derives from (r_sorted, phi,
 *            m_cum, G) into the workspace.  Non-zero: the caller states that the immediately
 *            preceding libhmc call on this workspace was hmc_orbit_turning_points with the same
 *            n, G, r_sorted, phi and m_cum and the same per-star inputs (contents unchanged), so the
 *            tables are still there and are not rebuilt, and the rejection bound F of every star,
 *            which that call also left in the workspace, is read instead of recomputed from two more
 *            table look-ups per star (same expressions, same bits).  Zero: always correct.
 */
HMC_API hmc_status hmc_sample_new_radius(uint64_t n, double G, uint64_t seed, uint32_t step,
        const double* r_sorted, const double* phi, const double* m_cum,
        const double* v_r, const double* v_t,
        const double* E, const double* J, const double* r_min, const double* r_max,
        const uint32_t* k_min, const uint32_t* k_max, const uint32_t* id,
        const uint8_t* star_status_in,
        double* r_new, double* v_r_new, double* v_t_new, uint16_t* n_try,
        uint8_t* star_status_out, uint64_t* counters, int32_t reuse_tables,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * hmc_sample_new_radius with the step number completed on the DEVICE: the Philox counter's step word (R9)
 * is step + step_dev[0], step_dev[0] read when the kernel runs.  This is what lets a CUDA graph captured from the
 * four calls of one orbit step be replayed: every other argument of a step is the same from one step to the next
 * (or alternates between two buffers), only the step number advances -- hmc_add_u32 enqueues word[0] += increment
 * on the stream, so a captured step can end by advancing its own counter.  Everything else as hmc_sample_new_radius
 * (PAPER.md:126-137); step_dev NULL: HMC_ERR_NULL.
 */
HMC_API hmc_status hmc_sample_new_radius_dstep(uint64_t n, double G, uint64_t seed, uint32_t step, const uint32_t* step_dev,
        const double* r_sorted, const double* phi, const double* m_cum,
        const double* v_r, const double* v_t,
        const double* E, const double* J, const double* r_min, const double* r_max,
        const uint32_t* k_min, const uint32_t* k_max, const uint32_t* id,
        const uint8_t* star_status_in,
        double* r_new, double* v_r_new, double* v_t_new, uint16_t* n_try,
        uint8_t* star_status_out, uint64_t* counters, int32_t reuse_tables,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

HMC_API hmc_status hmc_add_u32(uint32_t* word, uint32_t increment, void* cuda_stream);

/*
 * S3 + S4 in one launch (the two calls above fused).  Computes exactly what
 * hmc_orbit_turning_points followed by hmc_sample_new_radius compute, bit for bit, and writes every
 * output of both (E .. star_status are S3's, r_new .. star_status_out S4's): each warp solves 32 stars,
 * keeps their orbits on chip and draws their new radii, so S3's outputs are never read back and
 * searching and drawing warps share an SM.  Arguments as in the two calls.  Measured on B200 at N = 1e7 it is
 * SLOWER than the two calls (about 3 ms against 0.90 + 0.69 ms): it is kept for API completeness
 * and compared with the oracle in the tests; nothing else here uses it.
 */
HMC_API hmc_status hmc_orbit_step(uint64_t n, double G, uint64_t seed, uint32_t step,
        const double* r_sorted, const double* v_r, const double* v_t,
        const double* phi, const double* m_cum, const uint32_t* id,
        double* E, double* J, double* r_min, double* r_max,
        uint32_t* k_min, uint32_t* k_max, uint8_t* star_status,
        double* r_new, double* v_r_new, double* v_t_new, uint16_t* n_try,
        uint8_t* star_status_out, uint64_t* counters,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Energy correction for the time-varying potential (R18):
 * a star's new orbit was drawn in the potential Phi of the previous step; once the potential Phi' of the new
 * configuration is known its energy is changed by the work done by the changing potential,
 *     dE = 1/2 [ (Phi'(r_old) - Phi(r_old)) + (Phi'(r_new) - Phi(r_new)) ],
 * and both velocity components are scaled by the same factor so that v_r / v_t is preserved.  With the shell
 * potential this leaves T + W of the whole cluster exactly unchanged over the step.
 * Call it after hmc_sort_by_radius and hmc_potential of the NEW configuration, before hmc_orbit_turning_points.
 * All arrays are [n] in the new sorted order (star k at node k):
 *   r_sorted, phi, m_cum   the new table; Phi'(r_new) of star k is phi[k]
 *   E_old                  the star's energy in the old potential (E of the previous step's S3)
 *   r_old, phi_old         its previous radius and the old potential there (previous step's r_sorted and phi
 *                          at its then node)            -- these three travel through the sort as columns
 *   v_r, v_t               the velocities the previous step's S4 gave it
 *   v_r_out, v_t_out       corrected velocities; star_status_out: 0, or HMC_STAR_NOKINETIC when the corrected
 *                          kinetic energy is not positive (velocities copied through, counted)
 * Phi(r_new) is taken from the draw's energy identity, Phi(r_new) = E_old - (v_r^2 + v_t^2)/2.
 */
HMC_API hmc_status hmc_energy_correction(uint64_t n, double G,
        const double* r_sorted, const double* phi, const double* m_cum,
        const double* E_old, const double* r_old, const double* phi_old,
        const double* v_r, const double* v_t,
        double* v_r_out, double* v_t_out, uint8_t* star_status_out, uint64_t* counters,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Diagnostics on the radius-sorted arrays (PAPER.md:140 "half-mass radius ..."; :346 Eq. 20; :354
 * total energy; R15-R17).  out is a DEVICE array of HMC_DIAG_LAGRANGE + nfrac doubles:
 *   out[HMC_DIAG_M]      M_N, total mass
 *   out[HMC_DIAG_T]      T = sum_k m_k (v_r^2 + v_t^2) / 2          (exact sum of the binary64 terms, rounded once)
 *   out[HMC_DIAG_W]      W = sum_k m_k Phi_k / 2                    (likewise; Phi_k includes the star's own term)
 *   out[HMC_DIAG_ETOT]   T + W
 *   out[HMC_DIAG_VIRIAL] 2 T / |W|
 *   out[HMC_DIAG_RH]     half-mass radius: r_k of the first star with M_k >= M_N / 2
 *   out[HMC_DIAG_TRH]    0.138 N / ln(0.1 N) * (r_h^3 / (G M_N))^(1/2)   (Eq. 20)
 *   out[HMC_DIAG_LAGRANGE + i]  Lagrange radius of mass_fractions[i]: r_k of the first star with
 *                        M_k >= mass_fractions[i] * M_N (the outermost star if there is none)
 * mass_fractions is a HOST array of nfrac values, 0 <= nfrac <= HMC_DIAG_MAX_FRACTIONS (may be NULL if 0).
 * Preconditions: m >= 0 (M_cum ascending), n >= 1.
 */
#define HMC_DIAG_MAX_FRACTIONS 16
enum { HMC_DIAG_M = 0, HMC_DIAG_T, HMC_DIAG_W, HMC_DIAG_ETOT, HMC_DIAG_VIRIAL, HMC_DIAG_RH, HMC_DIAG_TRH, HMC_DIAG_LAGRANGE };

HMC_API hmc_status hmc_diagnostics(uint64_t n, double G,
        const double* r_sorted, const double* v_r, const double* v_t, const double* m_sorted,
        const double* phi, const double* m_cum,
        int32_t nfrac, const double* mass_fractions, double* out,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Relaxation: the two steps of the paper's loop between the potential and the new orbits.
 *
 * hmc_relaxation_timestep -- Eq. 7 on radial bins of HMC_BIN = 20 consecutive sorted stars
 * (the n mod 20 stars left over join the last bin), and "the minimum is taken as the value of the
 * global relaxation timestep" (:108):
 *     T_b = (theta_max / (pi/2)) (pi/32) <v_rel>^3 / ( ln(gamma n) G^2 n_b <(M_1 + M_2)^2> )
 * over the bin's neighbour pairs (2j, 2j+1): v_rel = ((v_r1 - v_r2)^2 + v_t1^2 + v_t2^2)^(1/2) (rms over the unknown
 * angle between the transverse velocities), n_b = stars of the bin / volume of the shell from the previous bin's last
 * star to this bin's last star (R19).  t_rel_bin: DEVICE [max(1, n / 20)] or NULL; t_rel_min: DEVICE [1]
 * (+inf when there is no pair).  gamma: the Coulomb logarithm's factor (the paper uses 0.1, :348).
 *
 * hmc_two_body_relaxation -- "an analytic expression for a representative encounter between two nearest-neighbor
 * stars" (the expression is in Joshi et al. 2000, not in the paper: DESIGN.md R20 is Henon's scheme).
 * Each pair (2j, 2j+1) undergoes one elastic encounter in its centre-of-mass frame by the deflection angle beta with
 * sin^2(beta/2) = 2 pi G^2 (m_1+m_2)^2 n_b ln(gamma n) dt / w^3 (capped at 1), about a uniformly random axis; the
 * pair's momentum and kinetic energy are conserved.  Where that expression has no value -- infinite n_b (a bin of
 * zero volume) times dt = 0, or a dt that is not finite -- the pair has no encounter (R20a).  The angles are Philox4x32-10(counter = (id of the pair's first
 * star, 1, step, t), key = seed), turned into unit vectors without trigonometric functions.  v_r_out / v_t_out [n]
 * receive the new velocities (an odd last star is copied).  Needs no workspace.  The step is dt, or, when dt_device
 * (DEVICE [1], e.g. t_rel_min of hmc_relaxation_timestep) is not NULL, dt * (*dt_device): no host round trip.
 */
#define HMC_BIN 20

HMC_API hmc_status hmc_relaxation_timestep(uint64_t n, double G, double gamma, double theta_max,
        const double* r_sorted, const double* v_r, const double* v_t, const double* m_sorted,
        double* t_rel_bin, double* t_rel_min,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

HMC_API hmc_status hmc_two_body_relaxation(uint64_t n, double G, double gamma, double dt, const double* dt_device,
        uint64_t seed, uint32_t step,
        const double* r_sorted, const double* v_r, const double* v_t, const double* m_sorted, const uint32_t* id,
        double* v_r_out, double* v_t_out, void* cuda_stream);

/*
 * Sharded step (SURVEY.md 8(e), 8(f) item 5; PAPER.md:196 duplicated arrays, :213-223 parallel flow, :239-243 sample
 * sort, :259-261 redistribution).  The stars are cut into `nranks` consecutive ranges of the sorted order, one per
 * GPU (Eq. 17's decomposition; host logic in paper_1206_5878_b200/shard.py).  Each rank sorts its stars
 * (hmc_sort_by_radius), places the splitters in its sorted radii (hmc_partition_points), exchanges partitions and
 * sorts what it received (hmc_sort_by_radius again: stable, so ties keep source order); then
 *   hmc_potential_totals   totals[4] (DEVICE, 32-byte aligned) = the shard's sum of m and of fl(m/r), each as a
 *                          double-double (hi, lo) pair: what the other shards need from this one
 *   hmc_potential_shard    as hmc_potential on the shard's stars, with rank_totals[nranks][4] (DEVICE: every shard's
 *                          totals, all-gathered) giving what lies before (lower ranks) and after (higher ranks):
 *                          M_k and S_k are the same exact sums rounded once as on one GPU (R1p)
 *   hmc_orbit_turning_points_range / hmc_sample_new_radius_range
 *                          S3 / S4 for the stars at positions first .. first+count-1 of the all-gathered table:
 *                          r_sorted, phi, m_cum are the TABLE's arrays [n]; v_r, v_t, id, every other per-star input
 *                          and every output are the range's own arrays [count].  first = 0, count = n is exactly
 *                          hmc_orbit_turning_points / hmc_sample_new_radius.  Workspace: hmc_workspace_bytes(n).
 *                          reuse_tables: the preceding S3 call on the workspace must have covered this range.
 * hmc_partition_points: counts[j] = number of radii <= splitters[j], j < nsplit (splitters, counts: DEVICE arrays).
 * Errors: HMC_ERR_SIZE if rank >= nranks, or first + count > n.
 */
HMC_API hmc_status hmc_potential_totals(uint64_t n, const double* r_sorted, const double* m_sorted, double* totals,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

HMC_API hmc_status hmc_potential_shard(uint64_t n, double G, const double* r_sorted, const double* m_sorted,
        uint32_t nranks, uint32_t rank, const double* rank_totals, double* phi, double* m_cum,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * hmc_potential_shard fused with the all-gather of the replicated table ("we maintain a copy of it on
 * all nodes"): besides phi and m_cum of its own shard, the launch stores the shard's r, phi and m_cum to npeers
 * further destinations, tile by tile as the scan produces them, so the exchange overlaps the arithmetic instead of
 * following it.  peer_r, peer_phi, peer_m_cum: HOST arrays of npeers DEVICE pointers, each pointing at this shard's
 * place (element `first` of that copy of the table); the memory may belong to another GPU (peer access over NVLink:
 * plain stores) or to this one.  A copy is complete when every rank's call has finished: the caller orders that
 * (a barrier across ranks, or stream order when the shards share a device).  npeers <= HMC_MAX_PEERS, else HMC_ERR_SIZE.
 */
HMC_API hmc_status hmc_potential_shard_push(uint64_t n, double G, const double* r_sorted, const double* m_sorted,
        uint32_t nranks, uint32_t rank, const double* rank_totals, double* phi, double* m_cum,
        int32_t npeers, double* const* peer_r, double* const* peer_phi, double* const* peer_m_cum,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

HMC_API hmc_status hmc_partition_points(uint64_t n, const double* r_sorted, uint32_t nsplit, const double* splitters,
        uint64_t* counts, void* cuda_stream);

HMC_API hmc_status hmc_orbit_turning_points_range(uint64_t n, uint64_t first, uint64_t count, double G,
        const double* r_sorted, const double* v_r, const double* v_t,
        const double* phi, const double* m_cum,
        double* E, double* J, double* r_min, double* r_max,
        uint32_t* k_min, uint32_t* k_max, uint8_t* star_status,
        uint64_t* counters,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The table build of S3 / S4 as a call of its own, and S3 on tables already built.  Every hmc_orbit_turning_points
 * call starts by deriving its search tables (node table, coarse table, radius directory: DESIGN.md section 4) from
 * (r_sorted, phi, m_cum) into the workspace; hmc_orbit_build_tables does just that, and
 * hmc_orbit_turning_points_prebuilt is hmc_orbit_turning_points_range without it (the tables in the workspace must be
 * those of the same r_sorted, phi, m_cum, G).  The pair computes exactly what the one call computes, with the same two
 * launches; it exists so that the ranges of a table can be searched without rebuilding it, and so that bench.py can
 * put a CUDA event between the two launches and time turning_points_kernel by itself.
 */
HMC_API hmc_status hmc_orbit_build_tables(uint64_t n, double G, const double* r_sorted, const double* phi, const double* m_cum,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

HMC_API hmc_status hmc_orbit_turning_points_prebuilt(uint64_t n, uint64_t first, uint64_t count, double G,
        const double* r_sorted, const double* v_r, const double* v_t,
        const double* phi, const double* m_cum,
        double* E, double* J, double* r_min, double* r_max,
        uint32_t* k_min, uint32_t* k_max, uint8_t* star_status,
        uint64_t* counters,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

HMC_API hmc_status hmc_sample_new_radius_range(uint64_t n, uint64_t first, uint64_t count, double G, uint64_t seed, uint32_t step,
        const double* r_sorted, const double* phi, const double* m_cum,
        const double* v_r, const double* v_t,
        const double* E, const double* J, const double* r_min, const double* r_max,
        const uint32_t* k_min, const uint32_t* k_max, const uint32_t* id,
        const uint8_t* star_status_in,
        double* r_new, double* v_r_new, double* v_t_new, uint16_t* n_try,
        uint8_t* star_status_out, uint64_t* counters, int32_t reuse_tables,
        void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Host-buffer variant of one whole orbit step (the four calls above, in order), for callers
 * whose star data lives in HOST memory.  r, v_r, v_t, m, id are HOST arrays [n] (unsorted);
 * r_new, v_r_new, v_t_new, m_out, id_out are HOST arrays [n] receiving the stars in radius-sorted
 * order of the INPUT radii.  Host buffers should be page-locked for the copies to be asynchronous.
 * `device_arena` is a DEVICE buffer of at least hmc_step_host_arena_bytes(n) bytes (256-byte
 * aligned) holding the staged columns, every intermediate and the workspace.
 * The call enqueues the copies in on `cuda_stream`, the four stages on a library-owned stream and the copies out on
 * another (the only state the library keeps: two streams and a few events per host thread and device, created at
 * first use), chained by events so that the three overlap: the sort starts when the radii have arrived, the sorted
 * masses and ids go back while the velocities are still coming in, and the new coordinates go back range by range
 * behind the draw.  `cuda_stream` waits for all of it: the host arrays are valid after the caller synchronises that
 * stream.  counters_host (HOST uint64[HMC_NCOUNTERS], may be NULL) receives the step's counters.
 */
HMC_API size_t hmc_step_host_arena_bytes(uint64_t n);

HMC_API hmc_status hmc_step_host(uint64_t n, double G, uint64_t seed, uint32_t step,
        const double* r, const double* v_r, const double* v_t, const double* m, const uint32_t* id,
        double* r_new, double* v_r_new, double* v_t_new, double* m_out, uint32_t* id_out,
        uint64_t* counters_host,
        void* device_arena, size_t arena_bytes, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* HMC_H */
