// mr_defer.cuh -- S6 on meshes far larger than L2: the DEFERRED tally (sm_100a).
//
// On a 512^3 mesh the fp64 tally is 1.07 GB against 126 MB of L2: the one atomic per segment of the plain cast
// kernel (red.global.add.f64 into the cell the ray happens to cross) misses L2 almost every time, and a miss costs a
// 128-byte DRAM line in and a 32-byte sector out for 8 useful bytes.  A batch touches every tally line about 40
// times, so the traffic is avoidable if the adds to one REGION of the tally are made while that region is in L2.
//
//   phase A  cast_defer_kernel: S1..S5 exactly as cast_kernel (same walker, records, score_terms), but S6 does not
//            touch the tally: the (cell, score) pair is appended to the BIN of the cell's region (bin = cell >> s,
//            a contiguous range of the linear cell index of at most L2/8 bytes of tally).  Every lane stages its own
//            pairs in shared memory (kDeferLane of them: a ray stays in one region for many steps) and writes them out
//            with 32-byte stores into the range of kDeferRange entries its WARP holds in that bin; a spent range costs
//            one global atomic; chunks of kDeferChunk entries come from a pool (lazily, taken by the warp that reserves
//            a chunk's first range).
//   phase B  defer_scatter_kernel: bin after bin, streams the pairs and adds them to the tally -- the same
//            red.global.add.f64, now into a region that stays in L2; DRAM sees the pairs once out and once in
//            (12 B each way) and every tally line once in and once out per batch.
// Nothing observable changes: tally[c] receives the same scores, in a different order (reading Q18).  If the pool
// runs out a warp adds its staged pairs straight to the tally (slow, always correct) and the host grows the pool.
//
// The kernel is persistent (lanes refill from a work counter, as rz_kernel does): a warp's reserved ranges and
// staged pairs are flushed and padded once, when the warp runs out of rays, not once per 32 rays.
#pragma once
#include "mr_device.cuh"

namespace mr {

constexpr int kDeferBins = 64;            // most regions the tally is cut into
constexpr int kDeferLane = 8;             // pairs a lane stages in shared memory before it writes them out
constexpr int kDeferRange = 128;          // entries a warp reserves in a bin at a time (multiple of kDeferLane)
constexpr int kDeferChunk = 4096;         // entries per pool chunk (multiple of kDeferRange)
constexpr unsigned kDeferNoCell = 0xffffffffu;   // padding entry
constexpr unsigned kDeferNoRange = 0xffffffffu;  // the warp holds no range in this bin yet
constexpr unsigned kDeferDirect = 0xfffffffeu;   // no chunk to be had (pool or chunk table exhausted): add straight to the tally

struct DeferParams {
    int bin_shift;                 // bin = cell >> bin_shift
    int nbin;
    int max_chunks;                // chunk-table entries per bin
    int pool_chunks;               // chunks in the pool
    uint32_t *cells;               // [pool_chunks * kDeferChunk]
    double *scores;                // [pool_chunks * kDeferChunk]
    int *table;                    // [nbin * max_chunks]: pool chunk of a bin's k-th chunk; -1 not allocated yet, -2 none (pool exhausted)
    unsigned long long *cursor;    // [nbin] entries reserved so far (multiples of kDeferRange)
    unsigned int *pool_next;       // chunks handed out (runs past pool_chunks when the pool is exhausted)
    unsigned long long *work;      // next ray of the persistent phase-A kernel
    unsigned long long *direct;    // pairs that took the slow path (pool exhausted)
    unsigned int *queue;           // phase B: next (bin, chunk) work item
};

// Staging per warp.  A ray's consecutive cells mostly lie in one region (a region is several mesh planes thick), so
// every LANE stages its own pairs -- kDeferLane of them, in its own shared-memory column -- and writes them out with
// vector stores when the column is full or the ray moves to another region; the space comes from the range of
// kDeferRange entries the WARP holds in that bin (a shared-memory atomic), and only a spent range costs a global atomic.
//   bytes per warp: scores 8 x kDeferLane x 32 | cells 4 x kDeferLane x 32 | pos[nbin] | used[nbin]
__host__ __device__ constexpr size_t defer_warp_smem_bytes(int nbin) { return ((size_t)kDeferLane * 32 * 12 + (size_t)nbin * 8 + 15) & ~(size_t)15; }

struct WarpBins {
    double *scores;    // [kDeferLane][32]
    unsigned *cells;   // [kDeferLane][32]
    unsigned *pos;     // [nbin] pool index of the warp's range in the bin (kDeferNoRange / kDeferDirect)
    unsigned *used;    // [nbin] entries of that range handed to lanes (runs past kDeferRange when it is spent)
};

__device__ __forceinline__ WarpBins warp_bins(unsigned char *base, int nbin)
{
    WarpBins wb;
    wb.scores = reinterpret_cast<double *>(base);
    wb.cells = reinterpret_cast<unsigned *>(base + (size_t)kDeferLane * 32 * 8);
    wb.pos = wb.cells + kDeferLane * 32;
    wb.used = wb.pos + nbin;
    return wb;
}

__device__ __forceinline__ int ld_volatile_s32(const int *p)
{
    int v;
    asm volatile("ld.volatile.global.s32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}

// 32-byte streaming accesses: the pairs are written once and read once, gigabytes apart -- they bypass L1 and are the
// first to leave L2 (STG/LDG.E.NA.EFL2.256; the L2::evict_first qualifier exists for 256-bit accesses only)
__device__ __forceinline__ void stg_stream_u8(void *p, uint4 a, uint4 b)
{
    asm volatile("st.global.L1::no_allocate.L2::evict_first.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(a.x), "r"(a.y),
                 "r"(a.z), "r"(a.w), "r"(b.x), "r"(b.y), "r"(b.z), "r"(b.w) : "memory");
}
__device__ __forceinline__ void stg_stream_d4(void *p, double a, double b, double c, double d)
{
    asm volatile("st.global.L1::no_allocate.L2::evict_first.v4.b64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}
__device__ __forceinline__ uint32_t ldg_stream_u32(const void *p)
{
    uint32_t v;
    asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ double ldg_stream_f64(const void *p)
{
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void ldg_stream_u8(const void *p, uint4 &a, uint4 &b)
{
    asm volatile("ld.global.nc.L1::no_allocate.L2::evict_first.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w), "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(p));
}
__device__ __forceinline__ void ldg_stream_d4(const void *p, double &a, double &b, double &c, double &d)
{
    asm volatile("ld.global.nc.L1::no_allocate.L2::evict_first.v4.b64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}

// All 32 lanes: the warp's range in bin b is spent (`used_true` entries of it were handed out): pad the rest, reserve
// the next one.  The warp that reserves a chunk's first range takes the chunk from the pool.
__device__ __forceinline__ void defer_new_range(const DeferParams &D, const WarpBins &wb, int b, unsigned used_true)
{
    const unsigned full = 0xffffffffu;
    const unsigned lane = threadIdx.x & 31;
    const unsigned pos = wb.pos[b];
    if (pos == kDeferDirect) {                                     // stays direct for the rest of the launch
        __syncwarp();
        if (lane == 0) wb.used[b] = 0;
        __syncwarp();
        return;
    }
    if (pos != kDeferNoRange)
        for (unsigned i = used_true + lane; i < (unsigned)kDeferRange; i += 32) D.cells[pos + i] = kDeferNoCell;
    unsigned npos = kDeferDirect;
    if (lane == 0) {
        const unsigned long long p = atomicAdd(D.cursor + b, (unsigned long long)kDeferRange);
        const unsigned long long k = p / kDeferChunk;
        const unsigned off = (unsigned)(p % kDeferChunk);
        int id = -2;
        if (k < (unsigned long long)D.max_chunks) {
            int *slot = D.table + (size_t)b * D.max_chunks + k;
            if (off == 0) {
                const unsigned got = atomicAdd(D.pool_next, 1u);
                id = got < (unsigned)D.pool_chunks ? (int)got : -2;
                *reinterpret_cast<volatile int *>(slot) = id;
                __threadfence();
            } else {
                while ((id = ld_volatile_s32(slot)) == -1) {}       // the allocating warp is between its two atomics
            }
        }
        if (id >= 0) npos = (unsigned)id * kDeferChunk + off;
    }
    npos = __shfl_sync(full, npos, 0);
    __syncwarp();
    if (lane == 0) {
        wb.pos[b] = npos;
        wb.used[b] = 0;
    }
    __syncwarp();
}

// All 32 lanes, every kDeferLane walk steps: every lane writes out the k (<= kDeferLane) pairs of its column into ONE
// 8-entry slot (32-byte aligned; padded) of the range the warp holds in the bin of the column's FIRST pair.  The pairs
// of a column are consecutive cells of one ray (lanes are refilled between windows only); where the ray crosses into
// the next region inside the window, up to kDeferLane - 1 pairs land in the neighbouring bin.  That costs nothing in
// correctness -- phase B adds every pair to tally[cell] whatever bin it sits in -- and next to nothing in locality: the
// neighbouring region is the one phase B works on just before or just after.
__device__ __forceinline__ void defer_write_out(const DeferParams &D, const WarpBins &wb, int k, double *tally)
{
    const unsigned full = 0xffffffffu;
    const unsigned lane = threadIdx.x & 31;
    const bool want = k > 0;
    if (!__ballot_sync(full, want)) return;
    const int bin = want ? (int)(wb.cells[lane] >> D.bin_shift) : 0;
    unsigned dst = kDeferDirect, u = 0;
    bool got = !want;
    for (;;) {
        if (!got) {
            const unsigned p = wb.pos[bin];
            u = atomicAdd(wb.used + bin, (unsigned)kDeferLane);
            if (p == kDeferDirect) { dst = kDeferDirect; got = true; }
            else if (p != kDeferNoRange && u + kDeferLane <= (unsigned)kDeferRange) { dst = p + u; got = true; }
        }
        unsigned fail = __ballot_sync(full, !got);
        if (!fail) break;
        while (fail) {                                             // ranges that are spent (or were never reserved)
            const int b = __shfl_sync(full, bin, __ffs(fail) - 1);
            const bool mine = !got && bin == b;
            const unsigned used_true = min(__reduce_min_sync(full, mine ? u : 0xffffffffu), (unsigned)kDeferRange);
            defer_new_range(D, wb, b, used_true);
            fail &= ~__ballot_sync(full, mine);
        }
    }
    if (want) {
        if (dst != kDeferDirect) {
            // rows >= k hold pairs of earlier windows: their cells are written as kDeferNoCell, their scores are never read
            uint4 c0, c1;
            c0.x = wb.cells[lane];
            c0.y = 1 < k ? wb.cells[1 * 32 + lane] : kDeferNoCell;
            c0.z = 2 < k ? wb.cells[2 * 32 + lane] : kDeferNoCell;
            c0.w = 3 < k ? wb.cells[3 * 32 + lane] : kDeferNoCell;
            c1.x = 4 < k ? wb.cells[4 * 32 + lane] : kDeferNoCell;
            c1.y = 5 < k ? wb.cells[5 * 32 + lane] : kDeferNoCell;
            c1.z = 6 < k ? wb.cells[6 * 32 + lane] : kDeferNoCell;
            c1.w = 7 < k ? wb.cells[7 * 32 + lane] : kDeferNoCell;
            stg_stream_u8(D.cells + dst, c0, c1);
            stg_stream_d4(D.scores + dst, wb.scores[lane], wb.scores[1 * 32 + lane], wb.scores[2 * 32 + lane], wb.scores[3 * 32 + lane]);
            if (k > 4)
                stg_stream_d4(D.scores + dst + 4, wb.scores[4 * 32 + lane], wb.scores[5 * 32 + lane], wb.scores[6 * 32 + lane],
                              wb.scores[7 * 32 + lane]);
        } else {
            for (int j = 0; j < k; ++j) red_add_f64(tally + wb.cells[j * 32 + lane], wb.scores[j * 32 + lane]);
            atomicAdd(D.direct, (unsigned long long)k);
        }
    }
}

// All 32 lanes, when the warp has no rays left: pad the ranges the warp still holds.
__device__ __forceinline__ void defer_drain(const DeferParams &D, const WarpBins &wb)
{
    const unsigned lane = threadIdx.x & 31;
    __syncwarp();
    for (int b = 0; b < D.nbin; ++b) {
        const unsigned pos = wb.pos[b], used = min(wb.used[b], (unsigned)kDeferRange);
        if (pos != kDeferNoRange && pos != kDeferDirect)
            for (unsigned i = used + lane; i < (unsigned)kDeferRange; i += 32) D.cells[pos + i] = kDeferNoCell;
    }
}

// ------------------------------------------------------------------------------------------------
// Phase A.  One lane per ray at a time, persistent; MIXED mode only (Real = float).
//   dynamic shared memory: [edges (EDGES_SHARED only)] [walker: 3 x blockDim x 16 B] [sigma: (M+N) x blockDim floats]
//                          [per warp: defer_warp_smem_bytes(nbin)]
// ------------------------------------------------------------------------------------------------
constexpr int kDeferRefillLanes = 4;

template <typename Rec, int EDGE_MODE>
__global__ void __launch_bounds__(128) cast_defer_kernel(const __grid_constant__ CastParams P, const __grid_constant__ DeferParams D)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int stride = blockDim.x;
    unsigned char *sp = smem_raw;
    double *s_edges = reinterpret_cast<double *>(sp);
    if (EDGE_MODE == EDGES_SHARED) sp += edges_smem_bytes_for(P.mesh.nedges);
    AxisF *axf = reinterpret_cast<AxisF *>(sp) + threadIdx.x;
    sp += sizeof(AxisF) * 3 * stride;
    float *sig = reinterpret_cast<float *>(sp) + threadIdx.x;
    sp += (sizeof(float) * (size_t)(P.M + P.N) * stride + 15) & ~(size_t)15;
    const WarpBins wb = warp_bins(sp + (threadIdx.x >> 5) * defer_warp_smem_bytes(D.nbin), D.nbin);
    const double *e = (EDGE_MODE == EDGES_SHARED) ? s_edges : P.mesh.edges;
    if (EDGE_MODE == EDGES_SHARED) {
        for (int i = threadIdx.x; i < P.mesh.nedges; i += blockDim.x) s_edges[i] = __ldg(P.mesh.edges + i);
    }
    const unsigned full = 0xffffffffu;
    const unsigned lane = threadIdx.x & 31;
    for (int b = lane; b < D.nbin; b += 32) {
        wb.pos[b] = kDeferNoRange;
        wb.used[b] = kDeferRange;                                  // spent: the first write-out reserves a range
    }
    __syncthreads();

    bool active = false, exhausted = false;
    Walker w{};
    Rec rec;
    double wa = 0.0;
    unsigned n_acc = 0, n_rej = 0;
    unsigned long long n_seg = 0;
    auto fetch = [&]() {
        if constexpr (Rec::kCoarse)
            rec.load_coarse(P.crecs, P.cshift, P.cnx, P.cny, walker_cell_index(w.pl0, w.dc0), walker_cell_index(w.pl1, w.dc1),
                            walker_cell_index(w.pl2, w.dc2));
        else
            rec.load(P.recs, P.ids, P.K, w.c);
    };
    for (;;) {
        // refill idle lanes (once per kDeferLane steps)
        const unsigned idle = __ballot_sync(full, !active);
        if (!exhausted && idle && (__popc(idle) >= kDeferRefillLanes || idle == full)) {
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(D.work, (unsigned long long)__popc(idle));
            base = __shfl_sync(full, base, 0);
            exhausted = (long long)(base + __popc(idle)) >= P.n;
            if (!active) {
                const long long i = (long long)base + __popc(idle & ((1u << lane) - 1u));
                if (i < P.n) {
                    const long long r = P.perm ? (long long)__ldg(P.perm + i) : i;
                    const Ray<float> R = load_ray<float>(P.rays, r);
                    const bool accepted = R.finite && (R.E > 0.f) && walker_init<EDGE_MODE>(w, axf, stride, P.mesh, e, R.o, R.d);
                    if (accepted) {
                        sigma_all<float>(P.xs, P.M, P.N, P.mix_off, P.mix_nuc, P.mix_w, R.E, sig, stride);
                        wa = R.W;
                        rec.reset();
                        fetch();
                        active = true;
                        ++n_acc;
                    } else
                        ++n_rej;
                }
            }
        }
        if (__ballot_sync(full, active) == 0) {
            if (exhausted) break;
            continue;
        }
        // kDeferLane walk steps; every scored segment goes into the lane's column
        int k = 0;
#pragma unroll 1
        for (int j = 0; j < kDeferLane; ++j) {
            if (active) {
                int cell;
                double len;
                const bool leave = walker_step<EDGE_MODE>(w, axf, stride, P.mesh, e, cell, len);
                const typename Rec::Value cur = rec.value();
                if (!leave) fetch();
                const double S = (double)Rec::sigma(cur, sig, stride, P.K);
                double g, ex;
                score_terms<false>(S, len, g, ex);
                if (len > 0.0) {                                   // a zero-length segment scores exactly 0
                    wb.cells[k * 32 + lane] = (unsigned)cell;
                    wb.scores[k * 32 + lane] = wa * g;
                    ++k;
                }
                wa *= ex;
                ++n_seg;
                active = !leave;
            }
        }
        defer_write_out(D, wb, k, P.tally);
    }
    defer_drain(D, wb);

    unsigned acc = n_acc, rej = n_rej;
    unsigned long long segs = n_seg;
    for (int o = 16; o > 0; o >>= 1) {
        acc += __shfl_xor_sync(full, acc, o);
        rej += __shfl_xor_sync(full, rej, o);
        segs += __shfl_xor_sync(full, segs, o);
    }
    if (lane == 0) {
        if (acc) atomicAdd(P.counters + 0, (unsigned long long)acc);
        if (rej) atomicAdd(P.counters + 1, (unsigned long long)rej);
        if (segs) atomicAdd(P.counters + 2, segs);
    }
}

// ------------------------------------------------------------------------------------------------
// Phase B.  Work items are the chunks, bin after bin, handed out by one counter: the chunks in flight at any time are
// consecutive, so the CTAs resident together add into one region of the tally (two where a bin ends).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) defer_scatter_kernel(const DeferParams D, double *__restrict__ tally)
{
    __shared__ unsigned s_first[kDeferBins + 1];
    __shared__ unsigned s_item;
    if (threadIdx.x == 0) {
        unsigned run = 0;
        for (int b = 0; b < D.nbin; ++b) {
            s_first[b] = run;
            run += (unsigned)min((D.cursor[b] + kDeferChunk - 1) / kDeferChunk, (unsigned long long)D.max_chunks);
        }
        s_first[D.nbin] = run;
    }
    __syncthreads();
    const unsigned total = s_first[D.nbin];
    for (;;) {
        if (threadIdx.x == 0) s_item = atomicAdd(D.queue, 1u);
        __syncthreads();
        const unsigned item = s_item;
        __syncthreads();
        if (item >= total) break;
        int b = 0;
        while (s_first[b + 1] <= item) ++b;
        const unsigned long long k = item - s_first[b];
        const int id = D.table[(size_t)b * D.max_chunks + k];
        if (id < 0) continue;
        const unsigned cnt = (unsigned)min((unsigned long long)kDeferChunk, D.cursor[b] - k * kDeferChunk);   // a multiple of kDeferRange
        const uint32_t *cells = D.cells + (size_t)id * kDeferChunk;
        const double *scores = D.scores + (size_t)id * kDeferChunk;
        // One entry per lane: a write-out slot holds 8 CONSECUTIVE cells of one ray, so 8 neighbouring lanes of an add
        // instruction carry neighbouring cells (x steps share a 32-byte sector of the tally): fewer L2 requests than
        // entries, where a lane adding its own slot entry by entry would make every add a request of its own.
        for (unsigned i = threadIdx.x; i < cnt; i += blockDim.x) {
            const uint32_t cell = ldg_stream_u32(cells + i);
            if (cell != kDeferNoCell) red_add_f64(tally + cell, ldg_stream_f64(scores + i));
        }
    }
}

}  // namespace mr
