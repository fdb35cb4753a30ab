// probe_random_access.cu -- what a random table look-up costs on this GPU (stand-alone; not part of libhmc).
//
// S3 and S4 end in a few random reads of the node table per star ("random accesses to the
// gravitational potential profile").  How those reads should be issued -- and from which N on the turning-point
// search goes by lane pairs (HMC_S3_PAIRS_MIN_N in hmc_orbit.cu) -- follows from four measurements made here:
//
//   1. size    : random 32-byte reads per ns against the table size (64 MB .. 3.2 GB), one, two (same 64-byte
//                half-line, two load instructions) and four (whole 128-byte line, four instructions) per look-up.
//   2. coop    : the same 64 / 128 bytes fetched by 2 / 4 LANES in ONE load instruction.
//   3. pages   : an L2-resident working set (64 KB per 2 MB page) spread over 16 .. 1600 pages: where the TLB ends.
//   4. revisit : a second, DEPENDENT read of the same line / same page / another page right after the first.
//
// Build and run:  python -m paper_1206_5878_b200.build --probe  &&  ./paper_1206_5878_b200/probe_random_access
// Every kernel runs 148 x 1024 threads, each with K = 64 dependent rounds (the address of a round depends on the
// data of the previous one), so what is printed is throughput under the latency of a full chip, not peak issue.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

static constexpr int K = 64;
static constexpr int CTAS = 148, THREADS = 1024;

__device__ __forceinline__ uint64_t mix(uint64_t x)
{
    x ^= x >> 33; x *= 0xff51afd7ed558ccdULL; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ULL; x ^= x >> 33;
    return x;
}

// one 32-byte sector, the load S3 / S4 use for a node
__device__ __forceinline__ double ld32(const char* p)
{
    double x, y, z, w;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(x), "=d"(y), "=d"(z), "=d"(w) : "l"(p));
    return x + w;
}

// SECTORS consecutive sectors per look-up, each by its own load instruction of the same lane
template <int SECTORS>
__global__ void __launch_bounds__(THREADS, 1) by_one_lane(const char* tab, uint64_t nslots, double* out)
{
    uint64_t s = mix(blockIdx.x * (uint64_t)THREADS + threadIdx.x + 12345);
    double acc = 0;
    for (int k = 0; k < K; ++k) {
        s = mix(s + (uint64_t)(acc != 1.2345));
        const uint64_t slot = (s % nslots) & ~(uint64_t)(SECTORS - 1);
#pragma unroll
        for (int i = 0; i < SECTORS; ++i) acc += ld32(tab + (slot + i) * 32);
    }
    if (acc == 1.2345) out[0] = acc;
}

// the same bytes by GROUP lanes in one load instruction (lanes of a group share the look-up)
template <int GROUP>
__global__ void __launch_bounds__(THREADS, 1) by_lane_group(const char* tab, uint64_t nslots, double* out)
{
    const uint32_t lane = threadIdx.x & 31;
    uint64_t s = mix((blockIdx.x * (uint64_t)THREADS + threadIdx.x) / GROUP + 12345);
    double acc = 0;
    for (int k = 0; k < K; ++k) {
        s = mix(s + (uint64_t)(acc != 1.2345));
        const uint64_t slot = (s % nslots) & ~(uint64_t)(GROUP - 1);
        acc += ld32(tab + (slot + (lane & (GROUP - 1))) * 32);
        acc += __shfl_xor_sync(0xffffffffu, acc, 1) * 1e-300;     // the group's lanes stay together
    }
    if (acc == 1.2345) out[0] = acc;
}

// npages pages of 2 MB; inside page p only the 64 KB chunk number hash(p) % 32 is touched
__global__ void __launch_bounds__(THREADS, 1) scattered(const char* tab, uint32_t npages, double* out)
{
    uint64_t s = mix(blockIdx.x * (uint64_t)THREADS + threadIdx.x + 999);
    double acc = 0;
    for (int k = 0; k < K; ++k) {
        s = mix(s + (uint64_t)(acc != 1.2345));
        const uint32_t page = (uint32_t)(s % npages);
        const uint64_t off = (uint64_t)page * (2u << 20) + (uint64_t)(mix(page) & 31) * 65536 + ((s >> 32) & 2047) * 32;
        acc += ld32(tab + off);
    }
    if (acc == 1.2345) out[0] = acc;
}

// MODE 0: one read per round; 1: then a dependent read of the other sector of the same 64 bytes; 2: of a random
// line of the same 2 MB page; 3: of another random page
template <int MODE>
__global__ void __launch_bounds__(THREADS, 1) revisit(const char* tab, uint64_t nslots, double* out)
{
    uint64_t s = mix(blockIdx.x * (uint64_t)THREADS + threadIdx.x + 777);
    double acc = 0;
    for (int k = 0; k < K; ++k) {
        s = mix(s + (uint64_t)(acc != 1.2345));
        const uint64_t slot = s % nslots;
        const double a = ld32(tab + slot * 32);
        acc += a;
        if (MODE > 0) {
            const uint64_t t = mix(s ^ 0x9e37) + (uint64_t)(a != 1.2345) - 1;      // depends on the first read
            uint64_t slot2 = MODE == 1 ? (slot ^ 1) : MODE == 2 ? ((slot & ~65535ull) | (t & 65535ull)) : t % nslots;
            if (slot2 >= nslots) slot2 = slot;
            acc += ld32(tab + slot2 * 32);
        }
    }
    if (acc == 1.2345) out[0] = acc;
}

template <class F>
static double per_ns(F launch, double lookups)
{
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    launch(); launch();
    cudaEventRecord(e0); launch(); cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return lookups / (ms * 1e6);
}

int main()
{
    double* out;
    cudaMalloc(&out, 8);
    const double threads = (double)CTAS * THREADS * K;
    const uint64_t sizes[4] = { 64000000ull, 320000000ull, 640000000ull, 3200000000ull };
    printf("look-ups per ns, %d x %d threads, %d dependent rounds each\n", CTAS, THREADS, K);
    printf("1. size / 2. coop: %-8s | %-28s | %-22s\n", "", "one lane: 32 B, 2x32 B, 4x32 B", "one instruction: 2 lanes 64 B, 4 lanes 128 B");
    for (uint64_t bytes : sizes) {
        char* tab;
        if (cudaMalloc(&tab, bytes) != cudaSuccess) { printf("cudaMalloc(%llu) failed\n", (unsigned long long)bytes); return 1; }
        cudaMemset(tab, 0, bytes);
        const uint64_t ns = bytes / 32;
        const double a = per_ns([&] { by_one_lane<1><<<CTAS, THREADS>>>(tab, ns, out); }, threads);
        const double b = per_ns([&] { by_one_lane<2><<<CTAS, THREADS>>>(tab, ns, out); }, threads);
        const double c = per_ns([&] { by_one_lane<4><<<CTAS, THREADS>>>(tab, ns, out); }, threads);
        const double d = per_ns([&] { by_lane_group<2><<<CTAS, THREADS>>>(tab, ns, out); }, threads / 2);
        const double e = per_ns([&] { by_lane_group<4><<<CTAS, THREADS>>>(tab, ns, out); }, threads / 4);
        printf("   table %5.0f MB          | %6.1f %6.1f %6.1f         | %6.1f %6.1f\n", bytes / 1e6, a, b, c, d, e);
        const double r0 = per_ns([&] { revisit<0><<<CTAS, THREADS>>>(tab, ns, out); }, threads);
        const double r1 = per_ns([&] { revisit<1><<<CTAS, THREADS>>>(tab, ns, out); }, threads);
        const double r2 = per_ns([&] { revisit<2><<<CTAS, THREADS>>>(tab, ns, out); }, threads);
        const double r3 = per_ns([&] { revisit<3><<<CTAS, THREADS>>>(tab, ns, out); }, threads);
        printf("4. revisit %5.0f MB: rounds per ns: single %.1f | + same 64 B %.1f | + same page %.1f | + other page %.1f\n",
               bytes / 1e6, r0, r1, r2, r3);
        cudaFree(tab);
    }
    {
        const uint64_t bytes = 3400000000ull;
        char* tab;
        if (cudaMalloc(&tab, bytes) != cudaSuccess) { printf("cudaMalloc failed\n"); return 1; }
        cudaMemset(tab, 0, bytes);
        const uint32_t pages[10] = { 16, 32, 64, 96, 128, 192, 256, 512, 1024, 1600 };
        for (uint32_t np : pages)
            printf("3. pages: %4u pages x 64 KB (%5.1f MB touched): %6.1f\n", np, np * 65536 / 1e6,
                   per_ns([&] { scattered<<<CTAS, THREADS>>>(tab, np, out); }, threads));
        cudaFree(tab);
    }
    return 0;
}
