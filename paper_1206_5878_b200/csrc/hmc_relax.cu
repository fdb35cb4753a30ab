// hmc_relax.cu -- relaxation timestep (Eq. 7; bins of 20 stars, :194) and two-body relaxation on
// neighbour pairs: SURVEY.md 8(f) item 3.  The step of the paper's loop that comes immediately
// before "new orbits"; embarrassingly parallel on the radius-sorted arrays.  The paper defers the expression of the
// representative encounter to Joshi et al. (2000); what is computed here is DESIGN.md R19 (timestep) and R20
// (encounter), whose statement is the oracle's source text.  Every operation is +, -, *, / or sqrt in the order
// written there (-fmad=false), so the results are compared bit for bit.
#include "hmc_common.cuh"

namespace hmc {

static constexpr uint32_t BIN = 20;                        // stars per radial bin
#define HMC_FOUR_PI_3 4.1887902047863909846
#define HMC_PI_OVER_2 1.5707963267948966192
#define HMC_PI_OVER_32 0.098174770424681038702
#define HMC_TWO_PI 6.2831853071795864769

__host__ __device__ __forceinline__ uint32_t n_bins(uint32_t n) { return n < BIN ? (n ? 1u : 0u) : n / BIN; }

// count / volume of the shell between the last star of the previous bin (r = 0 for the first) and the bin's last star
__device__ __forceinline__ double bin_density(uint32_t n, const double* __restrict__ r, uint32_t b, uint32_t nb)
{
    const uint32_t first = b * BIN, last = (b + 1 == nb) ? n - 1 : first + BIN - 1;
    const double r_in = b ? __ldg(r + first - 1) : 0.0, r_out = __ldg(r + last);
    const double vol = HMC_FOUR_PI_3 * ((r_out * r_out) * r_out - (r_in * r_in) * r_in);
    return (double)(last - first + 1) / vol;
}

// one thread per bin: the sums over a bin's pairs run in pair order
__global__ void __launch_bounds__(256)
relaxation_timestep_kernel(uint32_t n, double G, double ln_gamma_n, double theta_max, const double* __restrict__ r,
                           const double* __restrict__ v_r, const double* __restrict__ v_t, const double* __restrict__ m,
                           double* __restrict__ t_bin)
{
    const uint32_t nb = n_bins(n);
    const uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb) return;
    const uint32_t first = b * BIN, last = (b + 1 == nb) ? n - 1 : first + BIN - 1;
    double sv = 0.0, sm = 0.0;
    uint32_t pairs = 0;
    for (uint32_t a = first; a + 1 <= last; a += 2) {
        const double dvr = __ldg(v_r + a) - __ldg(v_r + a + 1);
        const double t1 = __ldg(v_t + a), t2 = __ldg(v_t + a + 1);
        const double w = sqrt(dvr * dvr + t1 * t1 + t2 * t2);
        const double M = __ldg(m + a) + __ldg(m + a + 1);
        sv += w; sm += M * M;
        ++pairs;
    }
    double T = __longlong_as_double(0x7ff0000000000000ll);
    if (pairs) {
        const double vmean = sv / (double)pairs, m2mean = sm / (double)pairs;
        const double dens = bin_density(n, r, b, nb);
        const double den = ((ln_gamma_n * (G * G)) * dens) * m2mean;
        if (den > 0.0) T = (((theta_max / HMC_PI_OVER_2) * HMC_PI_OVER_32) * ((vmean * vmean) * vmean)) / den;
    }
    t_bin[b] = T;
}

// minimum over the bins, one CTA ("the minimum is taken as the value of the global relaxation timestep")
__global__ void __launch_bounds__(1024) min_timestep_kernel(const double* __restrict__ t_bin, uint32_t nb, double* __restrict__ out)
{
    __shared__ double sh[32];
    double best = __longlong_as_double(0x7ff0000000000000ll);
    for (uint32_t b = threadIdx.x; b < nb; b += blockDim.x) { const double T = t_bin[b]; if (T < best) best = T; }
    for (int d = 16; d > 0; d >>= 1) { const double o = __shfl_xor_sync(0xffffffffu, best, d); if (o < best) best = o; }
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 32; ++w) if (sh[w] < best) best = sh[w];
        *out = best;
    }
}

// (cos, sin) of a uniform angle without trigonometric functions: a uniform point (a, b) of the unit disc by rejection,
// then the doubled angle ((a^2 - b^2) / s, 2ab / s), s = a^2 + b^2.  Draw t uses Philox counter (id, 1, step, t).
__device__ __forceinline__ void unit_vector(uint32_t id, uint32_t step, uint32_t k0, uint32_t k1, uint32_t& t, double& c, double& s_out)
{
    while (t < 64u) {
        uint32_t w[4];
        philox4x32_10(id, 1u, step, t, k0, k1, w);
        ++t;
        const double a = 2.0 * u53_to_unit(w[0], w[1]) - 1.0;
        const double b = 2.0 * u53_to_unit(w[2], w[3]) - 1.0;
        const double s = a * a + b * b;
        if (s > 0.0 && s < 1.0) { c = (a * a - b * b) / s; s_out = (2.0 * (a * b)) / s; return; }
    }
    c = 1.0; s_out = 0.0;
}

// one thread per pair of neighbours (2j, 2j+1)
__global__ void __launch_bounds__(256)
two_body_relaxation_kernel(uint32_t n, double G, double ln_gamma_n, double dt_in, const double* __restrict__ dt_dev,
                           uint32_t k0, uint32_t k1, uint32_t step,
                           const double* __restrict__ r, const double* __restrict__ v_r, const double* __restrict__ v_t,
                           const double* __restrict__ m, const uint32_t* __restrict__ id, double* __restrict__ v_r_out,
                           double* __restrict__ v_t_out)
{
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t a = 2 * j, b = a + 1;
    if (a >= n) return;
    if (b >= n) { v_r_out[a] = v_r[a]; v_t_out[a] = v_t[a]; return; }              // odd star out
    const double dt = dt_dev ? dt_in * __ldg(dt_dev) : dt_in;                      // a device-resident step (T_rel of this step) times a factor
    const uint32_t nb = n_bins(n);
    uint32_t bin = a / BIN;
    if (bin >= nb) bin = nb - 1;
    const double dens = bin_density(n, r, bin, nb);
    const double2 mm = make_double2(__ldg(m + a), __ldg(m + b)), rr = make_double2(__ldg(v_r + a), __ldg(v_r + b)),
                  tt = make_double2(__ldg(v_t + a), __ldg(v_t + b));
    const double m1 = mm.x, m2 = mm.y, M = m1 + m2;
    uint32_t t = 0;
    double cphi, sphi, cpsi, spsi;
    const uint32_t sid = __ldg(id + a);
    unit_vector(sid, step, k0, k1, t, cphi, sphi);
    unit_vector(sid, step, k0, k1, t, cpsi, spsi);
    const double x1 = tt.x, z1 = rr.x;
    const double x2 = tt.y * cphi, y2 = tt.y * sphi, z2 = rr.y;
    const double wx = x1 - x2, wy = 0.0 - y2, wz = z1 - z2;
    const double wp2 = wx * wx + wy * wy, w2 = wp2 + wz * wz, wn = sqrt(w2);
    double2 out_r = rr, out_t = tt;
    if ((wn > 0.0) && (M > 0.0)) {
        double S = (((((HMC_TWO_PI * (G * G)) * (M * M)) * dens) * ln_gamma_n) * dt) / (w2 * wn);
        // R20a: no encounter where the expression has no value (S NaN: infinite density times dt = 0; or dt not finite)
        if (!(S == S) || !(dt < __longlong_as_double(0x7ff0000000000000ll))) S = 0.0;
        if (!(S < 1.0)) S = 1.0;
        if (!(S > 0.0)) S = 0.0;
        const double cb = 1.0 - 2.0 * S, sb = 2.0 * sqrt(S * (1.0 - S));
        const double wp = sqrt(wp2);
        double e1x, e1y, e1z, e2x, e2y, e2z;
        if (wp > 0.0) {
            e1x = wy / wp; e1y = (0.0 - wx) / wp; e1z = 0.0;
            const double q = wp * wn;
            e2x = (wx * wz) / q; e2y = (wy * wz) / q; e2z = (0.0 - wp2) / q;
        } else { e1x = 1.0; e1y = 0.0; e1z = 0.0; e2x = 0.0; e2y = 1.0; e2z = 0.0; }
        const double k = wn * sb;
        const double nx = wx * cb + k * (e1x * cpsi + e2x * spsi);
        const double ny = wy * cb + k * (e1y * cpsi + e2y * spsi);
        const double nz = wz * cb + k * (e1z * cpsi + e2z * spsi);
        const double Vx = (m1 * x1 + m2 * x2) / M, Vy = (m2 * y2) / M, Vz = (m1 * z1 + m2 * z2) / M;
        const double f1 = m2 / M, f2 = m1 / M;
        const double ax = Vx + f1 * nx, ay = Vy + f1 * ny, az = Vz + f1 * nz;
        const double bx = Vx - f2 * nx, by = Vy - f2 * ny, bz = Vz - f2 * nz;
        out_r = make_double2(az, bz);
        out_t = make_double2(sqrt(ax * ax + ay * ay), sqrt(bx * bx + by * by));
    }
    v_r_out[a] = out_r.x; v_r_out[b] = out_r.y;
    v_t_out[a] = out_t.x; v_t_out[b] = out_t.y;
}

hmc_status relaxation_timestep(uint64_t n, double G, double ln_gamma_n, double theta_max, const double* r, const double* v_r,
                               const double* v_t, const double* m, double* t_rel_bin, double* t_rel_min, const Workspace& ws,
                               cudaStream_t st)
{
    const uint32_t nb = n_bins((uint32_t)n);
    double* t_bin = t_rel_bin ? t_rel_bin : reinterpret_cast<double*>(ws.keys_alt);      // [n] doubles of scratch: plenty
    if (nb) {
        relaxation_timestep_kernel<<<(nb + 255) / 256, 256, 0, st>>>((uint32_t)n, G, ln_gamma_n, theta_max, r, v_r, v_t, m, t_bin);
        HMC_LAUNCH_CHECK();
    }
    min_timestep_kernel<<<1, 1024, 0, st>>>(t_bin, nb, t_rel_min);
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

hmc_status two_body_relaxation(uint64_t n, double G, double ln_gamma_n, double dt, const double* dt_dev, uint64_t seed, uint32_t step, const double* r,
                               const double* v_r, const double* v_t, const double* m, const uint32_t* id, double* v_r_out,
                               double* v_t_out, cudaStream_t st)
{
    const uint32_t pairs = (uint32_t)((n + 1) / 2);
    two_body_relaxation_kernel<<<(pairs + 255) / 256, 256, 0, st>>>((uint32_t)n, G, ln_gamma_n, dt, dt_dev, (uint32_t)seed,
                                                                    (uint32_t)(seed >> 32), step, r, v_r, v_t, m, id, v_r_out, v_t_out);
    HMC_LAUNCH_CHECK();
    return HMC_OK;
}

}  // namespace hmc
