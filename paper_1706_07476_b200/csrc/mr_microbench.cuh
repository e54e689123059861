// mr_microbench.cuh -- the L2 fp64-atomic ceiling the cast kernel is measured against (SURVEY.md §7 "Hard parts",
// §8(d) "L2 atomic throughput against a measured micro-benchmark").
//
// The cast kernel's lanes are 32 unrelated rays: per segment each lane issues one red.global.add.f64 into the cell it
// crosses and (on the plain-record path) one 16- or 32-byte record load from the same cell.  This kernel issues
// exactly that access pattern and nothing else: every lane adds 1.0 into a pseudo-random cell of an `ncell`-double
// array (L2-resident at 69 MB), optionally after loading `gather_bytes` from a record array at the same cell; lanes in
// groups of `group` (1, 2, 4, ...) take CONSECUTIVE cells, i.e. share a 32-byte sector when group = 4 -- what a
// warp-cooperative or spatially sorted walk would buy.  Result: lane-operations per second.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mr {

struct RedBenchParams {
    double *tally;          // [ncell]
    const uint4 *recs;      // [ncell * gather_bytes / 16] or null
    unsigned ncell;
    int group;              // lanes that take consecutive cells
    int gather_bytes;       // 0, 16 or 32
    int iters;              // operations per thread
    unsigned *sink;         // keeps the gathers alive
};

__device__ __forceinline__ unsigned rb_hash(unsigned x)
{
    x ^= x >> 16; x *= 0x7feb352du;
    x ^= x >> 15; x *= 0x846ca68bu;
    x ^= x >> 16;
    return x;
}

__global__ void __launch_bounds__(128) red_bench_kernel(const RedBenchParams P)
{
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned g = tid / P.group, within = tid % P.group;
    const unsigned ngroups_cells = P.ncell / P.group;
    unsigned acc = 0;
    for (int it = 0; it < P.iters; ++it) {
        const unsigned cell = (unsigned)(((unsigned long long)rb_hash(g * 0x9e3779b9u + it * 0x85ebca6bu + 1u) * ngroups_cells) >> 32) * P.group + within;
        if (P.gather_bytes == 16) {
            uint4 v;
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(P.recs + cell));
            acc += v.x ^ v.w;
        } else if (P.gather_bytes == 32) {
            uint4 a, b;
            asm volatile("ld.global.nc.L1::no_allocate.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w), "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(P.recs + 2 * (size_t)cell));
            acc += a.x ^ b.w;
        }
        asm volatile("red.global.add.f64 [%0], %1;" ::"l"(P.tally + cell), "d"(1.0) : "memory");
    }
    if (acc == 0x12345678u) *P.sink = acc;
}

}  // namespace mr
