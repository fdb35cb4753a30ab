// hmc_api.cu -- extern "C" boundary of libhmc (include/hmc.h): argument checks, workspace
// carve-up, stream plumbing.  No arithmetic of the method lives here.
#include <cmath>
#include <vector>
#include "hmc_common.cuh"

namespace hmc {

std::atomic<uint64_t> g_launches{ 0 };

int sm_count()
{
    static std::atomic<int> cached[64];                     // zero-initialised; one slot per device ordinal
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HMC_SM_COUNT_FALLBACK;
    const bool slot = dev >= 0 && dev < 64;
    if (slot && (sms = cached[dev].load(std::memory_order_relaxed)) > 0) return sms;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
        sms = HMC_SM_COUNT_FALLBACK;
    if (slot) cached[dev].store(sms, std::memory_order_relaxed);
    return sms;
}

static hmc_status check_ws(const void* ws, size_t bytes, uint64_t n)
{
    if (!ws) return HMC_ERR_WORKSPACE;
    if (misaligned(ws, 256)) return HMC_ERR_WORKSPACE;
    if (bytes < carve(nullptr, n).total) return HMC_ERR_WORKSPACE;
    return HMC_OK;
}

// arena of the host-buffer step: every device array the four stages touch
struct Arena {
    double *r, *vr, *vt, *m;             // staged inputs (unsorted)
    uint32_t* id;
    double *rs, *vrs, *vts, *ms;         // sorted
    uint32_t *ids, *perm;
    double *phi, *mcum, *E, *J, *rmin, *rmax;
    uint32_t *kmin, *kmax;
    uint8_t *st0, *st1;
    double *rn, *vrn, *vtn;
    uint64_t* counters;
    void* ws;
    size_t ws_bytes;
    size_t total;
};

static Arena carve_arena(void* base, uint64_t n)
{
    Arena a;
    char* p = static_cast<char*>(base);
    size_t off = 0;
    auto take = [&](size_t bytes) { char* q = p ? p + off : nullptr; off += align_up(bytes, 256); return q; };
    auto f64 = [&]() { return reinterpret_cast<double*>(take(n * 8)); };
    auto u32 = [&]() { return reinterpret_cast<uint32_t*>(take(n * 4)); };
    auto u8 = [&]() { return reinterpret_cast<uint8_t*>(take(n)); };
    a.r = f64(); a.vr = f64(); a.vt = f64(); a.m = f64(); a.id = u32();
    a.rs = f64(); a.vrs = f64(); a.vts = f64(); a.ms = f64(); a.ids = u32(); a.perm = u32();
    a.phi = f64(); a.mcum = f64(); a.E = f64(); a.J = f64(); a.rmin = f64(); a.rmax = f64();
    a.kmin = u32(); a.kmax = u32(); a.st0 = u8(); a.st1 = u8();
    a.rn = f64(); a.vrn = f64(); a.vtn = f64();
    a.counters = reinterpret_cast<uint64_t*>(take(HMC_NCOUNTERS * 8));
    a.ws_bytes = carve(nullptr, n).total;
    a.ws = take(a.ws_bytes);
    a.total = off;
    return a;
}

// hmc_step_host only: two library-owned streams and a few events, so that the three things a host-buffer step does --
// copy in (on the caller's stream), compute (on `kern`) and copy out (on `copy`) -- overlap: PCIe is full duplex and
// the step is bound by it.  One set per (host thread, device), created at first use and kept for the life of the
// thread: the only state the library owns.
static constexpr int HOST_CHUNKS = 4;     // ranges S4 is cut into so that the copy back starts behind the first of them

struct HostStepStreams {
    bool made = false;
    cudaStream_t kern = nullptr, copy = nullptr;
    cudaEvent_t r_up = nullptr, id_up = nullptr, vt_up = nullptr, mid_sorted = nullptr, done = nullptr;
    cudaEvent_t drawn[HOST_CHUNKS] = {};
};

static hmc_status host_step_streams(HostStepStreams** out)
{
    static thread_local std::vector<HostStepStreams> per_device;
    int dev = 0;
    HMC_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0) return HMC_ERR_CUDA;
    if ((size_t)dev >= per_device.size()) per_device.resize((size_t)dev + 1);
    HostStepStreams& hs = per_device[(size_t)dev];
    if (!hs.made) {
        HMC_CUDA_TRY(cudaStreamCreateWithFlags(&hs.kern, cudaStreamNonBlocking));
        HMC_CUDA_TRY(cudaStreamCreateWithFlags(&hs.copy, cudaStreamNonBlocking));
        cudaEvent_t* evs[] = { &hs.r_up, &hs.id_up, &hs.vt_up, &hs.mid_sorted, &hs.done };
        for (cudaEvent_t* e : evs) HMC_CUDA_TRY(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
        for (int c = 0; c < HOST_CHUNKS; ++c) HMC_CUDA_TRY(cudaEventCreateWithFlags(&hs.drawn[c], cudaEventDisableTiming));
        hs.made = true;
    }
    *out = &hs;
    return HMC_OK;
}

}  // namespace hmc

using namespace hmc;

#define REQUIRE_PTR(p)  do { if (!(p)) return HMC_ERR_NULL; } while (0)
#define REQUIRE_ALIGN(p, a) do { if (misaligned((p), (a))) return HMC_ERR_ALIGN; } while (0)

extern "C" {

size_t hmc_workspace_bytes(uint64_t n) { return carve(nullptr, n).total; }

int32_t hmc_version(void) { return 200; }

uint32_t hmc_t_max(void) { return HMC_T_MAX; }

uint64_t hmc_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

const char* hmc_status_string(hmc_status s)
{
    switch (s) {
        case HMC_OK: return "HMC_OK";
        case HMC_ERR_NULL: return "HMC_ERR_NULL: a required pointer is NULL";
        case HMC_ERR_SIZE: return "HMC_ERR_SIZE: n or ncols out of range";
        case HMC_ERR_WORKSPACE: return "HMC_ERR_WORKSPACE: workspace NULL, misaligned or too small";
        case HMC_ERR_ALIGN: return "HMC_ERR_ALIGN: array pointer not aligned to its element size";
        case HMC_ERR_CUDA: return "HMC_ERR_CUDA: CUDA runtime call or kernel launch failed";
        case HMC_ERR_STATIC_LIMIT:
            return "HMC_ERR_STATIC_LIMIT: n exceeds HMC_STATIC_MAX_N (2^24 stars), the capacity of the library's built-in "
                   "scratch array; use the call that takes a workspace";
        default: return "HMC: unknown status";
    }
}

hmc_status hmc_sort_by_radius(uint64_t n, const double* r_in, double* r_sorted, uint32_t* perm, int32_t ncols,
                              const double* const* cols_in, double* const* cols_out, const uint32_t* id_in,
                              uint32_t* id_out, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N || ncols < 0 || ncols > HMC_MAX_COLS) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(r_in); REQUIRE_PTR(r_sorted); REQUIRE_PTR(perm);
    if (ncols > 0) { REQUIRE_PTR(cols_in); REQUIRE_PTR(cols_out); }
    for (int c = 0; c < ncols; ++c) {
        REQUIRE_PTR(cols_in[c]); REQUIRE_PTR(cols_out[c]);
        REQUIRE_ALIGN(cols_in[c], 8); REQUIRE_ALIGN(cols_out[c], 8);
    }
    if ((id_in == nullptr) != (id_out == nullptr)) return HMC_ERR_NULL;
    REQUIRE_ALIGN(r_in, 8); REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(perm, 4);
    if (id_in) { REQUIRE_ALIGN(id_in, 4); REQUIRE_ALIGN(id_out, 4); }
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return sort_by_radius(n, r_in, r_sorted, perm, ncols, cols_in, cols_out, id_in, id_out, carve(workspace, n),
                          static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_potential(uint64_t n, double G, const double* r_sorted, const double* m_sorted, double* phi,
                         double* m_cum, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(m_sorted); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(m_sorted, 8); REQUIRE_ALIGN(phi, 8); REQUIRE_ALIGN(m_cum, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return potential(n, G, r_sorted, m_sorted, phi, m_cum, nullptr, 0, 0, carve(workspace, n), static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_orbit_turning_points(uint64_t n, double G, const double* r_sorted, const double* v_r,
                                    const double* v_t, const double* phi, const double* m_cum, double* E, double* J,
                                    double* r_min, double* r_max, uint32_t* k_min, uint32_t* k_max,
                                    uint8_t* star_status, uint64_t* counters, void* workspace,
                                    size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(v_r); REQUIRE_PTR(v_t); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum);
    REQUIRE_PTR(E); REQUIRE_PTR(J); REQUIRE_PTR(r_min); REQUIRE_PTR(r_max); REQUIRE_PTR(k_min); REQUIRE_PTR(k_max);
    REQUIRE_PTR(star_status);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(v_r, 8); REQUIRE_ALIGN(v_t, 8); REQUIRE_ALIGN(phi, 8);
    REQUIRE_ALIGN(m_cum, 8); REQUIRE_ALIGN(E, 8); REQUIRE_ALIGN(J, 8); REQUIRE_ALIGN(r_min, 8);
    REQUIRE_ALIGN(r_max, 8); REQUIRE_ALIGN(k_min, 4); REQUIRE_ALIGN(k_max, 4);
    if (counters) REQUIRE_ALIGN(counters, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return turning_points(n, 0, n, G, r_sorted, v_r, v_t, phi, m_cum, E, J, r_min, r_max, k_min, k_max, star_status,
                          counters, carve(workspace, n), static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_sample_new_radius(uint64_t n, double G, uint64_t seed, uint32_t step, const double* r_sorted,
                                 const double* phi, const double* m_cum, const double* v_r, const double* v_t,
                                 const double* E, const double* J, const double* r_min, const double* r_max,
                                 const uint32_t* k_min, const uint32_t* k_max, const uint32_t* id,
                                 const uint8_t* star_status_in, double* r_new, double* v_r_new, double* v_t_new,
                                 uint16_t* n_try, uint8_t* star_status_out, uint64_t* counters,
                                 int32_t reuse_tables, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum); REQUIRE_PTR(v_r); REQUIRE_PTR(v_t);
    REQUIRE_PTR(E); REQUIRE_PTR(J); REQUIRE_PTR(r_min); REQUIRE_PTR(r_max); REQUIRE_PTR(k_min); REQUIRE_PTR(k_max);
    REQUIRE_PTR(id); REQUIRE_PTR(star_status_in); REQUIRE_PTR(r_new); REQUIRE_PTR(v_r_new); REQUIRE_PTR(v_t_new);
    REQUIRE_PTR(star_status_out);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(phi, 8); REQUIRE_ALIGN(m_cum, 8); REQUIRE_ALIGN(v_r, 8);
    REQUIRE_ALIGN(v_t, 8); REQUIRE_ALIGN(E, 8); REQUIRE_ALIGN(J, 8); REQUIRE_ALIGN(r_min, 8); REQUIRE_ALIGN(r_max, 8);
    REQUIRE_ALIGN(k_min, 4); REQUIRE_ALIGN(k_max, 4); REQUIRE_ALIGN(id, 4); REQUIRE_ALIGN(r_new, 8);
    REQUIRE_ALIGN(v_r_new, 8); REQUIRE_ALIGN(v_t_new, 8);
    if (n_try) REQUIRE_ALIGN(n_try, 2);
    if (counters) REQUIRE_ALIGN(counters, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return sample_new_radius(n, 0, n, G, seed, step, r_sorted, phi, m_cum, v_r, v_t, E, J, r_min, r_max, k_min, k_max, id,
                             star_status_in, r_new, v_r_new, v_t_new, n_try, star_status_out, counters, reuse_tables != 0,
                             carve(workspace, n), static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_orbit_step(uint64_t n, double G, uint64_t seed, uint32_t step, const double* r_sorted,
                          const double* v_r, const double* v_t, const double* phi, const double* m_cum,
                          const uint32_t* id, double* E, double* J, double* r_min, double* r_max, uint32_t* k_min,
                          uint32_t* k_max, uint8_t* star_status, double* r_new, double* v_r_new, double* v_t_new,
                          uint16_t* n_try, uint8_t* star_status_out, uint64_t* counters, void* workspace,
                          size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(v_r); REQUIRE_PTR(v_t); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum); REQUIRE_PTR(id);
    REQUIRE_PTR(E); REQUIRE_PTR(J); REQUIRE_PTR(r_min); REQUIRE_PTR(r_max); REQUIRE_PTR(k_min); REQUIRE_PTR(k_max);
    REQUIRE_PTR(star_status); REQUIRE_PTR(r_new); REQUIRE_PTR(v_r_new); REQUIRE_PTR(v_t_new); REQUIRE_PTR(star_status_out);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(v_r, 8); REQUIRE_ALIGN(v_t, 8); REQUIRE_ALIGN(phi, 8); REQUIRE_ALIGN(m_cum, 8);
    REQUIRE_ALIGN(id, 4); REQUIRE_ALIGN(E, 8); REQUIRE_ALIGN(J, 8); REQUIRE_ALIGN(r_min, 8); REQUIRE_ALIGN(r_max, 8);
    REQUIRE_ALIGN(k_min, 4); REQUIRE_ALIGN(k_max, 4); REQUIRE_ALIGN(r_new, 8); REQUIRE_ALIGN(v_r_new, 8); REQUIRE_ALIGN(v_t_new, 8);
    if (n_try) REQUIRE_ALIGN(n_try, 2);
    if (counters) REQUIRE_ALIGN(counters, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return orbit_step(n, 0, n, G, seed, step, r_sorted, v_r, v_t, phi, m_cum, id, E, J, r_min, r_max, k_min, k_max, star_status,
                      r_new, v_r_new, v_t_new, n_try, star_status_out, counters, carve(workspace, n),
                      static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_energy_correction(uint64_t n, double G, const double* r_sorted, const double* phi, const double* m_cum,
                                 const double* E_old, const double* r_old, const double* phi_old, const double* v_r,
                                 const double* v_t, double* v_r_out, double* v_t_out, uint8_t* star_status_out,
                                 uint64_t* counters, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum); REQUIRE_PTR(E_old); REQUIRE_PTR(r_old); REQUIRE_PTR(phi_old);
    REQUIRE_PTR(v_r); REQUIRE_PTR(v_t); REQUIRE_PTR(v_r_out); REQUIRE_PTR(v_t_out); REQUIRE_PTR(star_status_out);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(phi, 8); REQUIRE_ALIGN(m_cum, 8); REQUIRE_ALIGN(E_old, 8); REQUIRE_ALIGN(r_old, 8);
    REQUIRE_ALIGN(phi_old, 8); REQUIRE_ALIGN(v_r, 8); REQUIRE_ALIGN(v_t, 8); REQUIRE_ALIGN(v_r_out, 8); REQUIRE_ALIGN(v_t_out, 8);
    if (counters) REQUIRE_ALIGN(counters, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return energy_correction(n, G, r_sorted, phi, m_cum, E_old, r_old, phi_old, v_r, v_t, v_r_out, v_t_out, star_status_out,
                             counters, carve(workspace, n), static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_diagnostics(uint64_t n, double G, const double* r_sorted, const double* v_r, const double* v_t,
                           const double* m_sorted, const double* phi, const double* m_cum, int32_t nfrac,
                           const double* mass_fractions, double* out, void* workspace, size_t workspace_bytes,
                           void* cuda_stream)
{
    if (n == 0 || n > HMC_MAX_N || nfrac < 0 || nfrac > HMC_DIAG_MAX_FRACTIONS) return HMC_ERR_SIZE;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(v_r); REQUIRE_PTR(v_t); REQUIRE_PTR(m_sorted); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum);
    REQUIRE_PTR(out);
    if (nfrac > 0) REQUIRE_PTR(mass_fractions);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(v_r, 8); REQUIRE_ALIGN(v_t, 8); REQUIRE_ALIGN(m_sorted, 8); REQUIRE_ALIGN(phi, 8);
    REQUIRE_ALIGN(m_cum, 8); REQUIRE_ALIGN(out, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return diagnostics(n, G, r_sorted, v_r, v_t, m_sorted, phi, m_cum, nfrac, mass_fractions, out, carve(workspace, n),
                       static_cast<cudaStream_t>(cuda_stream));
}

/* ---- relaxation (include/hmc.h "Relaxation") -------------------------------------------------------------------- */

hmc_status hmc_relaxation_timestep(uint64_t n, double G, double gamma, double theta_max, const double* r_sorted,
                                   const double* v_r, const double* v_t, const double* m_sorted, double* t_rel_bin,
                                   double* t_rel_min, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    REQUIRE_PTR(t_rel_min); REQUIRE_ALIGN(t_rel_min, 8);
    if (n > 0) { REQUIRE_PTR(r_sorted); REQUIRE_PTR(v_r); REQUIRE_PTR(v_t); REQUIRE_PTR(m_sorted); }
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(v_r, 8); REQUIRE_ALIGN(v_t, 8); REQUIRE_ALIGN(m_sorted, 8);
    if (t_rel_bin) REQUIRE_ALIGN(t_rel_bin, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    const double lg = std::log(gamma * (double)n);               // the Coulomb logarithm ln(gamma N), once, on the host
    return relaxation_timestep(n, G, lg, theta_max, r_sorted, v_r, v_t, m_sorted, t_rel_bin, t_rel_min, carve(workspace, n),
                               static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_two_body_relaxation(uint64_t n, double G, double gamma, double dt, const double* dt_device, uint64_t seed, uint32_t step,
                                   const double* r_sorted, const double* v_r, const double* v_t, const double* m_sorted,
                                   const uint32_t* id, double* v_r_out, double* v_t_out, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(v_r); REQUIRE_PTR(v_t); REQUIRE_PTR(m_sorted); REQUIRE_PTR(id);
    REQUIRE_PTR(v_r_out); REQUIRE_PTR(v_t_out);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(v_r, 8); REQUIRE_ALIGN(v_t, 8); REQUIRE_ALIGN(m_sorted, 8); REQUIRE_ALIGN(id, 4);
    REQUIRE_ALIGN(v_r_out, 8); REQUIRE_ALIGN(v_t_out, 8); REQUIRE_ALIGN(dt_device, 8);
    const double lg = std::log(gamma * (double)n);
    return two_body_relaxation(n, G, lg, dt, dt_device, seed, step, r_sorted, v_r, v_t, m_sorted, id, v_r_out, v_t_out,
                               static_cast<cudaStream_t>(cuda_stream));
}

/* ---- sharded step (include/hmc.h "Sharded step") ------------------------------------------------------------- */

hmc_status hmc_potential_totals(uint64_t n, const double* r_sorted, const double* m_sorted, double* totals,
                                void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    REQUIRE_PTR(totals); REQUIRE_ALIGN(totals, 32);
    if (n > 0) { REQUIRE_PTR(r_sorted); REQUIRE_PTR(m_sorted); REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(m_sorted, 8); }
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return potential_totals(n, r_sorted, m_sorted, totals, carve(workspace, n), static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_potential_shard(uint64_t n, double G, const double* r_sorted, const double* m_sorted, uint32_t nranks,
                               uint32_t rank, const double* rank_totals, double* phi, double* m_cum, void* workspace,
                               size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N || nranks == 0 || rank >= nranks) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(m_sorted); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum); REQUIRE_PTR(rank_totals);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(m_sorted, 8); REQUIRE_ALIGN(phi, 8); REQUIRE_ALIGN(m_cum, 8);
    REQUIRE_ALIGN(rank_totals, 32);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return potential(n, G, r_sorted, m_sorted, phi, m_cum, rank_totals, nranks, rank, carve(workspace, n),
                     static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_potential_shard_push(uint64_t n, double G, const double* r_sorted, const double* m_sorted, uint32_t nranks,
                                    uint32_t rank, const double* rank_totals, double* phi, double* m_cum, int32_t npeers,
                                    double* const* peer_r, double* const* peer_phi, double* const* peer_m_cum,
                                    void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N || nranks == 0 || rank >= nranks || npeers < 0 || npeers > HMC_MAX_PEERS) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(m_sorted); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum); REQUIRE_PTR(rank_totals);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(m_sorted, 8); REQUIRE_ALIGN(phi, 8); REQUIRE_ALIGN(m_cum, 8);
    REQUIRE_ALIGN(rank_totals, 32);
    if (npeers > 0) { REQUIRE_PTR(peer_r); REQUIRE_PTR(peer_phi); REQUIRE_PTR(peer_m_cum); }
    for (int g = 0; g < npeers; ++g) {
        REQUIRE_PTR(peer_r[g]); REQUIRE_PTR(peer_phi[g]); REQUIRE_PTR(peer_m_cum[g]);
        REQUIRE_ALIGN(peer_r[g], 8); REQUIRE_ALIGN(peer_phi[g], 8); REQUIRE_ALIGN(peer_m_cum[g], 8);
    }
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return potential(n, G, r_sorted, m_sorted, phi, m_cum, rank_totals, nranks, rank, carve(workspace, n),
                     static_cast<cudaStream_t>(cuda_stream), npeers, peer_r, peer_phi, peer_m_cum);
}

hmc_status hmc_partition_points(uint64_t n, const double* r_sorted, uint32_t nsplit, const double* splitters,
                                uint64_t* counts, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    if (nsplit == 0) return HMC_OK;
    REQUIRE_PTR(splitters); REQUIRE_PTR(counts);
    if (n > 0) REQUIRE_PTR(r_sorted);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(splitters, 8); REQUIRE_ALIGN(counts, 8);
    return partition_points(n, r_sorted, nsplit, splitters, counts, static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_orbit_turning_points_range(uint64_t n, uint64_t first, uint64_t count, double G, const double* r_sorted,
                                          const double* v_r, const double* v_t, const double* phi, const double* m_cum,
                                          double* E, double* J, double* r_min, double* r_max, uint32_t* k_min,
                                          uint32_t* k_max, uint8_t* star_status, uint64_t* counters, void* workspace,
                                          size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N || first > n || count > n - first) return HMC_ERR_SIZE;
    if (n == 0 || count == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(v_r); REQUIRE_PTR(v_t); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum);
    REQUIRE_PTR(E); REQUIRE_PTR(J); REQUIRE_PTR(r_min); REQUIRE_PTR(r_max); REQUIRE_PTR(k_min); REQUIRE_PTR(k_max);
    REQUIRE_PTR(star_status);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(v_r, 8); REQUIRE_ALIGN(v_t, 8); REQUIRE_ALIGN(phi, 8);
    REQUIRE_ALIGN(m_cum, 8); REQUIRE_ALIGN(E, 8); REQUIRE_ALIGN(J, 8); REQUIRE_ALIGN(r_min, 8);
    REQUIRE_ALIGN(r_max, 8); REQUIRE_ALIGN(k_min, 4); REQUIRE_ALIGN(k_max, 4);
    if (counters) REQUIRE_ALIGN(counters, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return turning_points(n, first, count, G, r_sorted, v_r, v_t, phi, m_cum, E, J, r_min, r_max, k_min, k_max, star_status,
                          counters, carve(workspace, n), static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_orbit_build_tables(uint64_t n, double G, const double* r_sorted, const double* phi, const double* m_cum,
                                  void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(phi, 8); REQUIRE_ALIGN(m_cum, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return orbit_build_tables(n, G, r_sorted, phi, m_cum, carve(workspace, n), static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_orbit_turning_points_prebuilt(uint64_t n, uint64_t first, uint64_t count, double G, const double* r_sorted,
                                          const double* v_r, const double* v_t, const double* phi, const double* m_cum,
                                          double* E, double* J, double* r_min, double* r_max, uint32_t* k_min,
                                          uint32_t* k_max, uint8_t* star_status, uint64_t* counters, void* workspace,
                                          size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N || first > n || count > n - first) return HMC_ERR_SIZE;
    if (n == 0 || count == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(v_r); REQUIRE_PTR(v_t); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum);
    REQUIRE_PTR(E); REQUIRE_PTR(J); REQUIRE_PTR(r_min); REQUIRE_PTR(r_max); REQUIRE_PTR(k_min); REQUIRE_PTR(k_max);
    REQUIRE_PTR(star_status);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(v_r, 8); REQUIRE_ALIGN(v_t, 8); REQUIRE_ALIGN(phi, 8);
    REQUIRE_ALIGN(m_cum, 8); REQUIRE_ALIGN(E, 8); REQUIRE_ALIGN(J, 8); REQUIRE_ALIGN(r_min, 8);
    REQUIRE_ALIGN(r_max, 8); REQUIRE_ALIGN(k_min, 4); REQUIRE_ALIGN(k_max, 4);
    if (counters) REQUIRE_ALIGN(counters, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return turning_points(n, first, count, G, r_sorted, v_r, v_t, phi, m_cum, E, J, r_min, r_max, k_min, k_max, star_status,
                          counters, carve(workspace, n), static_cast<cudaStream_t>(cuda_stream), true);
}

hmc_status hmc_sample_new_radius_range(uint64_t n, uint64_t first, uint64_t count, double G, uint64_t seed, uint32_t step,
                                       const double* r_sorted, const double* phi, const double* m_cum, const double* v_r,
                                       const double* v_t, const double* E, const double* J, const double* r_min,
                                       const double* r_max, const uint32_t* k_min, const uint32_t* k_max,
                                       const uint32_t* id, const uint8_t* star_status_in, double* r_new, double* v_r_new,
                                       double* v_t_new, uint16_t* n_try, uint8_t* star_status_out, uint64_t* counters,
                                       int32_t reuse_tables, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N || first > n || count > n - first) return HMC_ERR_SIZE;
    if (n == 0 || count == 0) return HMC_OK;
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum); REQUIRE_PTR(v_r); REQUIRE_PTR(v_t);
    REQUIRE_PTR(E); REQUIRE_PTR(J); REQUIRE_PTR(r_min); REQUIRE_PTR(r_max); REQUIRE_PTR(k_min); REQUIRE_PTR(k_max);
    REQUIRE_PTR(id); REQUIRE_PTR(star_status_in); REQUIRE_PTR(r_new); REQUIRE_PTR(v_r_new); REQUIRE_PTR(v_t_new);
    REQUIRE_PTR(star_status_out);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(phi, 8); REQUIRE_ALIGN(m_cum, 8); REQUIRE_ALIGN(v_r, 8);
    REQUIRE_ALIGN(v_t, 8); REQUIRE_ALIGN(E, 8); REQUIRE_ALIGN(J, 8); REQUIRE_ALIGN(r_min, 8); REQUIRE_ALIGN(r_max, 8);
    REQUIRE_ALIGN(k_min, 4); REQUIRE_ALIGN(k_max, 4); REQUIRE_ALIGN(id, 4); REQUIRE_ALIGN(r_new, 8);
    REQUIRE_ALIGN(v_r_new, 8); REQUIRE_ALIGN(v_t_new, 8);
    if (n_try) REQUIRE_ALIGN(n_try, 2);
    if (counters) REQUIRE_ALIGN(counters, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return sample_new_radius(n, first, count, G, seed, step, r_sorted, phi, m_cum, v_r, v_t, E, J, r_min, r_max, k_min, k_max,
                             id, star_status_in, r_new, v_r_new, v_t_new, n_try, star_status_out, counters, reuse_tables != 0,
                             carve(workspace, n), static_cast<cudaStream_t>(cuda_stream));
}

hmc_status hmc_sample_new_radius_dstep(uint64_t n, double G, uint64_t seed, uint32_t step, const uint32_t* step_dev,
                                       const double* r_sorted, const double* phi, const double* m_cum, const double* v_r,
                                       const double* v_t, const double* E, const double* J, const double* r_min,
                                       const double* r_max, const uint32_t* k_min, const uint32_t* k_max,
                                       const uint32_t* id, const uint8_t* star_status_in, double* r_new, double* v_r_new,
                                       double* v_t_new, uint16_t* n_try, uint8_t* star_status_out, uint64_t* counters,
                                       int32_t reuse_tables, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(step_dev); REQUIRE_ALIGN(step_dev, 4);
    REQUIRE_PTR(r_sorted); REQUIRE_PTR(phi); REQUIRE_PTR(m_cum); REQUIRE_PTR(v_r); REQUIRE_PTR(v_t);
    REQUIRE_PTR(E); REQUIRE_PTR(J); REQUIRE_PTR(r_min); REQUIRE_PTR(r_max); REQUIRE_PTR(k_min); REQUIRE_PTR(k_max);
    REQUIRE_PTR(id); REQUIRE_PTR(star_status_in); REQUIRE_PTR(r_new); REQUIRE_PTR(v_r_new); REQUIRE_PTR(v_t_new);
    REQUIRE_PTR(star_status_out);
    REQUIRE_ALIGN(r_sorted, 8); REQUIRE_ALIGN(phi, 8); REQUIRE_ALIGN(m_cum, 8); REQUIRE_ALIGN(v_r, 8);
    REQUIRE_ALIGN(v_t, 8); REQUIRE_ALIGN(E, 8); REQUIRE_ALIGN(J, 8); REQUIRE_ALIGN(r_min, 8); REQUIRE_ALIGN(r_max, 8);
    REQUIRE_ALIGN(k_min, 4); REQUIRE_ALIGN(k_max, 4); REQUIRE_ALIGN(id, 4); REQUIRE_ALIGN(r_new, 8);
    REQUIRE_ALIGN(v_r_new, 8); REQUIRE_ALIGN(v_t_new, 8);
    if (n_try) REQUIRE_ALIGN(n_try, 2);
    if (counters) REQUIRE_ALIGN(counters, 8);
    hmc_status s = check_ws(workspace, workspace_bytes, n);
    if (s != HMC_OK) return s;
    return sample_new_radius(n, 0, n, G, seed, step, r_sorted, phi, m_cum, v_r, v_t, E, J, r_min, r_max, k_min, k_max,
                             id, star_status_in, r_new, v_r_new, v_t_new, n_try, star_status_out, counters, reuse_tables != 0,
                             carve(workspace, n), static_cast<cudaStream_t>(cuda_stream), step_dev);
}

hmc_status hmc_add_u32(uint32_t* word, uint32_t increment, void* cuda_stream)
{
    REQUIRE_PTR(word); REQUIRE_ALIGN(word, 4);
    return add_u32(word, increment, static_cast<cudaStream_t>(cuda_stream));
}

size_t hmc_step_host_arena_bytes(uint64_t n) { return carve_arena(nullptr, n).total; }

hmc_status hmc_step_host(uint64_t n, double G, uint64_t seed, uint32_t step, const double* r, const double* v_r,
                         const double* v_t, const double* m, const uint32_t* id, double* r_new, double* v_r_new,
                         double* v_t_new, double* m_out, uint32_t* id_out, uint64_t* counters_host,
                         void* device_arena, size_t arena_bytes, void* cuda_stream)
{
    if (n > HMC_MAX_N) return HMC_ERR_SIZE;
    if (n == 0) return HMC_OK;
    REQUIRE_PTR(r); REQUIRE_PTR(v_r); REQUIRE_PTR(v_t); REQUIRE_PTR(m); REQUIRE_PTR(id);
    REQUIRE_PTR(r_new); REQUIRE_PTR(v_r_new); REQUIRE_PTR(v_t_new); REQUIRE_PTR(m_out); REQUIRE_PTR(id_out);
    if (!device_arena || misaligned(device_arena, 256)) return HMC_ERR_WORKSPACE;
    Arena a = carve_arena(device_arena, n);
    if (arena_bytes < a.total) return HMC_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    HostStepStreams* hs = nullptr;
    hmc_status s = host_step_streams(&hs);
    if (s != HMC_OK) return s;
    cudaStream_t K = hs->kern, D = hs->copy;
    // Everything is enqueued by `enqueue`; a failure part-way returns from it at once, and the code behind it then
    // still orders the caller's stream after whatever had been put on K and D by then (work that reads and writes
    // the arena and the host buffers), so a caller that reuses them after an error does not race with it.
    auto enqueue = [&]() -> hmc_status {
    // copy in, on the caller's stream, in the order the stages need the columns: r (the sort), m and id (they go
    // back to the host sorted, and S2 needs m), then the velocities (S3)
    HMC_CUDA_TRY(cudaMemcpyAsync(a.r, r, n * 8, cudaMemcpyHostToDevice, st));
    HMC_CUDA_TRY(cudaEventRecord(hs->r_up, st));
    HMC_CUDA_TRY(cudaMemcpyAsync(a.m, m, n * 8, cudaMemcpyHostToDevice, st));
    HMC_CUDA_TRY(cudaMemcpyAsync(a.id, id, n * 4, cudaMemcpyHostToDevice, st));
    HMC_CUDA_TRY(cudaEventRecord(hs->id_up, st));
    HMC_CUDA_TRY(cudaMemcpyAsync(a.vr, v_r, n * 8, cudaMemcpyHostToDevice, st));
    HMC_CUDA_TRY(cudaMemcpyAsync(a.vt, v_t, n * 8, cudaMemcpyHostToDevice, st));
    HMC_CUDA_TRY(cudaEventRecord(hs->vt_up, st));
    Workspace ws = carve(a.ws, n);
    // S1 as soon as the radii are there: the permutation and the sorted radii (no columns yet)
    HMC_CUDA_TRY(cudaStreamWaitEvent(K, hs->r_up, 0));
    HMC_CUDA_TRY(cudaMemsetAsync(a.counters, 0, HMC_NCOUNTERS * 8, K));
    s = sort_by_radius(n, a.r, a.rs, a.perm, 0, nullptr, nullptr, nullptr, nullptr, ws, K);
    if (s != HMC_OK) return s;
    // masses and ids follow the permutation and start back to the host while the velocities are still coming in
    HMC_CUDA_TRY(cudaStreamWaitEvent(K, hs->id_up, 0));
    {
        const double* cin[1] = { a.m };
        double* cout[1] = { a.ms };
        s = gather_by_perm(n, a.perm, 1, cin, cout, a.id, a.ids, K);
        if (s != HMC_OK) return s;
    }
    HMC_CUDA_TRY(cudaEventRecord(hs->mid_sorted, K));
    HMC_CUDA_TRY(cudaStreamWaitEvent(D, hs->mid_sorted, 0));
    HMC_CUDA_TRY(cudaMemcpyAsync(m_out, a.ms, n * 8, cudaMemcpyDeviceToHost, D));
    HMC_CUDA_TRY(cudaMemcpyAsync(id_out, a.ids, n * 4, cudaMemcpyDeviceToHost, D));
    s = potential(n, G, a.rs, a.ms, a.phi, a.mcum, nullptr, 0, 0, ws, K);
    if (s != HMC_OK) return s;
    HMC_CUDA_TRY(cudaStreamWaitEvent(K, hs->vt_up, 0));
    {
        const double* cin[2] = { a.vr, a.vt };
        double* cout[2] = { a.vrs, a.vts };
        s = gather_by_perm(n, a.perm, 2, cin, cout, nullptr, nullptr, K);
        if (s != HMC_OK) return s;
    }
    s = turning_points(n, 0, n, G, a.rs, a.vrs, a.vts, a.phi, a.mcum, a.E, a.J, a.rmin, a.rmax, a.kmin, a.kmax, a.st0,
                       a.counters, ws, K);
    if (s != HMC_OK) return s;
    // S4 in HOST_CHUNKS ranges of the sorted order; the new coordinates of a range start back to the host as soon as
    // its draw is done, while the next range is being drawn
    const uint64_t per = (n + HOST_CHUNKS - 1) / HOST_CHUNKS;
    for (int c = 0; c < HOST_CHUNKS; ++c) {
        const uint64_t first = umin64((uint64_t)c * per, n), count = umin64(per, n - first);
        if (count == 0) break;
        s = sample_new_radius(n, first, count, G, seed, step, a.rs, a.phi, a.mcum, a.vrs + first, a.vts + first, a.E + first,
                              a.J + first, a.rmin + first, a.rmax + first, a.kmin + first, a.kmax + first, a.ids + first,
                              a.st0 + first, a.rn + first, a.vrn + first, a.vtn + first, nullptr, a.st1 + first, a.counters,
                              true, ws, K);
        if (s != HMC_OK) return s;
        HMC_CUDA_TRY(cudaEventRecord(hs->drawn[c], K));
        HMC_CUDA_TRY(cudaStreamWaitEvent(D, hs->drawn[c], 0));
        HMC_CUDA_TRY(cudaMemcpyAsync(r_new + first, a.rn + first, count * 8, cudaMemcpyDeviceToHost, D));
        HMC_CUDA_TRY(cudaMemcpyAsync(v_r_new + first, a.vrn + first, count * 8, cudaMemcpyDeviceToHost, D));
        HMC_CUDA_TRY(cudaMemcpyAsync(v_t_new + first, a.vtn + first, count * 8, cudaMemcpyDeviceToHost, D));
    }
    if (counters_host)
        HMC_CUDA_TRY(cudaMemcpyAsync(counters_host, a.counters, HMC_NCOUNTERS * 8, cudaMemcpyDeviceToHost, D));
    HMC_CUDA_TRY(cudaEventRecord(hs->done, D));
    HMC_CUDA_TRY(cudaStreamWaitEvent(st, hs->done, 0));          // the caller's stream completes when everything is back
    return HMC_OK;
    };
    s = enqueue();
    if (s != HMC_OK) {                                           // error path only: K -> D -> the caller's stream
        if (cudaEventRecord(hs->drawn[0], K) == cudaSuccess) (void)cudaStreamWaitEvent(D, hs->drawn[0], 0);
        if (cudaEventRecord(hs->done, D) == cudaSuccess) (void)cudaStreamWaitEvent(st, hs->done, 0);
    }
    return s;
}

}  // extern "C"
