// monteray.cu -- host side of the C ABI declared in include/monteray.h.
//
// One translation unit: the context (device buffers, staging ring, options), argument
// checking, and the kernel launches.  Device code lives in mr_device.cuh.  Nothing here
// falls back to the CPU: without a CUDA device every entry point fails with MR_ERR_CUDA.
#include "../../include/monteray.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <condition_variable>
#include <memory>
#include <mutex>
#include <cstdio>
#include <cstring>
#include <string>
#include <thread>
#include <unordered_map>
#include <vector>

#define MR_PACK_MAX_SLOTS MR_MAX_SLOTS
#include "mr_device.cuh"
#include "mr_sort.cuh"
#include "mr_defer.cuh"
#include "mr_tiled.cuh"
#include "mr_microbench.cuh"

using namespace mr;

namespace {

thread_local std::string g_create_error;

constexpr int kStageSlots = 2;
constexpr size_t kEdgesSmemMax = 96 * 1024;  // larger meshes read their planes from global memory

struct DeviceGuard {
    int prev = -1;
    bool changed = false;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) changed = (cudaSetDevice(dev) == cudaSuccess);
    }
    ~DeviceGuard()
    {
        if (changed) cudaSetDevice(prev);
    }
};

}  // namespace

// Producer ring (mr_ring_*): `slots` page-locked buffers, each with a device buffer behind it.
struct RingSlot {
    enum State { FREE = 0, FILLING = 1, SHIPPING = 2, IN_FLIGHT = 3 };
    void *pinned = nullptr;
    void *d_buf = nullptr;
    cudaEvent_t ev_copied = nullptr;   // H2D out of `pinned` finished: the host buffer may be refilled
    cudaEvent_t ev_done = nullptr;     // kernels reading `d_buf` finished: the device buffer may be overwritten
    int state = FREE;                  // guarded by Ring::m
    int index = 0;                     // position in Ring::slots (and of d_buf in the ring's one device allocation)
    long long cursor = 0;              // rays reserved (guarded by Ring::m)
    std::atomic<long long> committed{0};   // rays whose copy into `pinned` has finished
};

struct Ring {
    std::mutex m;                      // slot states, cursors, `open`
    std::condition_variable cv;
    std::mutex ship_m;                 // serialises the CUDA calls that ship a slot
    std::vector<RingSlot *> slots;
    long long cap = 0;                 // rays per slot
    int open = 0;                      // slot being filled
    long long rays_pushed = 0, slots_shipped = 0;
    double wait_ms = 0.0;
    int error = MR_OK;                 // first error of a ship
    std::string error_msg;
    // Slot merging (guarded by ship_m).  The slots' device buffers are consecutive pieces of ONE allocation, so slots
    // whose copies are queued but whose cast is not -- the "pending" range, consecutive FULL slots that do not wrap -- are
    // cast by one ordering pre-pass and one launch over all their rays.
    void *d_all = nullptr;
    int pend_first = 0, pend_n = 0;
    long long pend_rays = 0;
    bool pend_full = true;             // every pending slot holds `cap` rays (a partial one must be the last)
    cudaEvent_t ev_cast = nullptr;     // behind the ring's latest cast on the context's stream
    bool cast_recorded = false;
    long long casts = 0;
};

struct mr_ctx {
    Ring *ring = nullptr;
    int device = 0;
    int precision = MR_PRECISION_MIXED;
    cudaStream_t stream = nullptr;
    cudaStream_t copy_stream = nullptr;
    // mr_read_tally_async: device snapshot of the tally, its own D2H stream and events
    cudaStream_t read_stream = nullptr;
    double *d_snap = nullptr;
    cudaEvent_t ev_snap = nullptr, ev_read = nullptr;
    bool read_pending = false;
    mr_allocator alloc{nullptr, nullptr, nullptr};
    std::string err;
    bool sticky_cuda = false;

    // mesh + tally
    int nx = 0, ny = 0, nz = 0, nedges = 0;
    long long ncell = 0;
    bool mesh_rz = false;              // R-Z mesh (mr_load_mesh_rz): nx = nr radial shells, ny = 1, x planes = radii
    bool mesh_sphere = false;          // with mesh_rz: 1-D spherical shells (mr_load_mesh_sphere), nz = 1
    bool mesh_arith = false;           // every plane position equals fma(p, h, e0) bit for bit
    double mesh_e0[3] = {0, 0, 0}, mesh_h[3] = {0, 0, 0};
    double *d_edges = nullptr;
    double *d_tally = nullptr;

    // materials
    int M = 0, K = 0, layout = 0;
    void *d_recs = nullptr;
    uint8_t *d_ids = nullptr;

    // tables: sigma per material; energy grids are shared between materials whose grids are bitwise identical
    struct Grid {
        std::vector<unsigned char> host;  // the grid as stored on the device (fp32 or fp64 bytes)
        void *d_E = nullptr;
        uint32_t *d_first = nullptr;      // bucket index, nb + 1 entries (XsDesc::first)
        uint32_t b0 = 0;
        int sh = 0, n = 0, refs = 0, id = 0;
    };
    std::vector<Grid *> grids;
    std::vector<Grid *> grid_of;          // [M]
    int next_grid_id = 0;
    std::vector<void *> d_S;
    std::vector<int> xs_n;
    XsDesc *d_xs = nullptr;
    bool xs_dirty = true;
    // nuclide tables and per-material mixtures (mr_load_nuclide_xs / mr_define_material)
    Grid *nuc_grid_of[MR_MAX_NUCLIDES] = {};
    void *nuc_S[MR_MAX_NUCLIDES] = {};
    int nuc_n[MR_MAX_NUCLIDES] = {};
    std::vector<std::vector<std::pair<int, double>>> mix;   // [M]: (nuclide, weight) list, empty = own table
    int N = 0;                             // nuclide slots in use by the resident descriptors (highest loaded index + 1)
    int *d_mix_off = nullptr, *d_mix_nuc = nullptr;
    void *d_mix_w = nullptr;

    unsigned long long *d_counters = nullptr;  // accepted, rejected, segments, spare | next-event: accepted, rejected, segments, spare

    // per-batch moments (allocated by the first mr_end_batch)
    double *d_prev = nullptr, *d_s2 = nullptr;
    long long nbatch = 0;

    // next-event detectors
    int ndet = 0;
    double *d_det = nullptr, *d_det_sum = nullptr;

    // host-batch staging ring
    void *pinned[kStageSlots] = {nullptr, nullptr};
    void *d_stage[kStageSlots] = {nullptr, nullptr};
    cudaEvent_t ev_copied[kStageSlots] = {nullptr, nullptr};
    cudaEvent_t ev_done[kStageSlots] = {nullptr, nullptr};
    size_t stage_cap_rays = 0;       // rays each slot can hold now
    long long stage_rays = 1 << 20;  // option MR_OPT_STAGE_RAYS (chunks grow from a quarter of it to twice it)
    int next_slot = 0;
    int copy_threads = 4;            // option MR_OPT_COPY_THREADS

    // Whole-batch staging for back-to-back host batches (run_batch): two device buffers that each hold a complete batch
    void *d_whole[2] = {nullptr, nullptr};
    size_t whole_cap_bytes = 0;
    cudaEvent_t ev_whole_copied = nullptr, ev_whole_done[2] = {nullptr, nullptr};
    int whole_next = 0;
    int ring_merge = 1;              // option MR_OPT_RING_MERGE: 0 one cast per slot, 1 auto (hold a slot back while an earlier ring cast runs), 2 hold until flush / wrap
    int whole_opt = 2;               // option MR_OPT_WHOLE_BATCH: 0 never, 1 always (pinned source), 2 auto = when the stream is still busy
    cudaEvent_t ev_t0 = nullptr, ev_t1 = nullptr;
    bool have_timing = false;
    std::vector<cudaEvent_t> kev;  // (start, stop) pairs around each cast-kernel launch of the last call
    size_t kev_used = 0;
    long long launches = 0;
    int block_threads = 128;
    int rz_block_threads = 256;      // R-Z / spherical cast kernel (option MR_OPT_RZ_BLOCK_THREADS)
    int sort_rays = 1;
    int pair_records = 1;            // option MR_OPT_PAIR_RECORDS

    // ray-ordering pre-pass scratch (grown on demand)
    // Two compute lanes: lane 0 queues on `stream`, lane 1 on the internal `stream2`.  Only the chunks of a HOST batch
    // alternate between them (run_batch), so that the ramp-down of one chunk's cast kernel overlaps the start of the
    // next chunk's; every other call works on lane 0.  Each lane has its own ordering scratch.
    int lane = 0;
    cudaStream_t stream2 = nullptr;
    cudaEvent_t ev_lane = nullptr;
    cudaStream_t work_stream() const { return lane ? stream2 : stream; }
    uint32_t *d_keys_l[2] = {nullptr, nullptr}, *d_perm_l[2] = {nullptr, nullptr}, *d_hist_l[2] = {nullptr, nullptr},
             *d_blk_hist_l[2] = {nullptr, nullptr};
    long long sort_cap_l[2] = {0, 0}, hist_cap_l[2] = {0, 0}, blk_hist_cap_l[2] = {0, 0};

    int order_mode = 0;              // option MR_OPT_ORDER_MODE: 0 auto, 1 slab-major, 2 longest first
    bool order_longest_auto = false; // set by cast_device: the deferred tally needs no slab locality, only a short tail
    // Tiled mixture index (K <= 3, MIXED, Cartesian): the distinct cell records as a small dictionary (shared memory in the
    // cast kernel) and a 2-byte index per cell stored in 4 x 4 (x, y) tiles of 32 bytes -- built by mr_load_materials when
    // the mesh has at most kDictMax distinct records (option MR_OPT_TILED_INDEX).
    int tiled_opt = 1;
    uint4 *d_dict = nullptr;
    uint4 *d_tiles = nullptr;
    int ndict = 0, ntx = 0, nty = 0, tile_bits = 16;
    // Tile-ordered score accumulators of the dictionary path (mr_tiled.cuh; option MR_OPT_TILED_TALLY): ntx * nty * nz tiles of
    // 64 / 32 / 16 doubles, moved into d_tally whenever the tally is looked at (flush_accumulators)
    int tiled_tally_opt = 0;
    double *d_tally_t = nullptr;
    long long tally_t_cells = 0;
    bool tiled_dirty = false;
    // mr_tally_device_ptr has handed d_tally out: from then on (until the next mesh) every cast adds straight into d_tally, so that
    // a view the caller keeps (an all-reduce buffer, a torch tensor) goes on following the tally -- no in-record / tile accumulators
    bool tally_borrowed = false;
    // Block-constant compositions (MIXED, K <= 4, Cartesian): one LAYOUT_K4 record per aligned block of 2^cshift cells per axis,
    // built by mr_load_materials when every such block holds one record (option MR_OPT_COARSE_RECORDS); cshift = 0: none
    int coarse_opt = 1;
    void *d_crecs = nullptr;
    int cshift = 0, cnx = 0, cny = 0, cnz = 0;
    // Deferred tally (mr_defer.cuh; option MR_OPT_DEFERRED_TALLY: 0 off, 1 on, 2 auto = coarse-record path on a mesh whose
    // tally exceeds twice the L2): pool of (cell, score) chunks, per-bin chunk table and the control words
    // ctl[0..63] bin cursors | ctl[64] chunks handed out | ctl[65] phase-A work counter | ctl[66] pairs added directly (cumulative) | ctl[67] phase-B work counter
    int defer_opt = 2;
    uint32_t *d_defer_cells = nullptr;
    double *d_defer_scores = nullptr;
    int *d_defer_table = nullptr;
    unsigned long long *d_defer_ctl = nullptr;
    unsigned long long *h_defer_ctl = nullptr;     // pinned: {chunks handed out, work, direct} after the last deferred cast
    cudaEvent_t ev_defer = nullptr;
    bool defer_pending = false;                    // h_defer_ctl is being written by the stream
    unsigned long long defer_direct_seen = 0;
    int defer_pool_chunks = 0, defer_max_chunks = 0;
    double defer_entries_per_ray = 0.0;            // sizing estimate; grows when a cast ran out of pool
    long long defer_pool_fixed = 0;                // option MR_OPT_DEFER_POOL_ENTRIES (0: sized by the estimate)
    int defer_shift_fixed = 0;                     // option MR_OPT_DEFER_REGION_SHIFT (0: from the L2 size)
    int coop_opt = 2;                // option MR_OPT_COOP_FLUSH: cast_coop_kernel (transposed tally adds) on the paths built for it;
                                     // 2 = auto: when tally + cell records fit in half the L2 (measured: config 5 6.05 -> 5.55 ms, config 2
                                     // 0.590 -> 0.558 ms; config 3, whose slabs stream through L2, 6.38 -> 7.22 ms: off there)
                                     // at every size: config 3 6.72 against 6.10 ms, config 2 0.62 against 0.57 ms, config 5 5.94 against 5.52 ms)
    int agg_first = 2;               // option MR_OPT_AGGREGATE_FIRST
    int fused_opt = 2;               // option MR_OPT_FUSED_TALLY: 0 off, 1 on, 2 auto (decided by mr_load_materials)
    bool fused = false;              // LAYOUT_K4 records carry the score accumulators (LAYOUT_K4F in the cast kernel)
    bool fused_dirty = false;        // in-record sums not yet moved into d_tally
    size_t l2_bytes = 0;             // device L2 size
    size_t rec_bytes_per_cell = 0;
    size_t resident_bytes() const { return (size_t)ncell * (8 + rec_bytes_per_cell); }   // tally + cell records

    size_t ray_bytes() const { return precision == MR_PRECISION_DOUBLE ? 64 : 32; }
    size_t real_bytes() const { return precision == MR_PRECISION_DOUBLE ? 8 : 4; }

    int fail(int code, const std::string &msg)
    {
        err = msg;
        return code;
    }
    int fail_cuda(cudaError_t e, const char *what)
    {
        sticky_cuda = true;
        err = std::string("CUDA error in ") + what + ": " + cudaGetErrorString(e);
        return e == cudaErrorMemoryAllocation ? MR_ERR_OOM : MR_ERR_CUDA;
    }
    void *dev_alloc(size_t bytes)
    {
        if (bytes == 0) bytes = 16;
        if (alloc.alloc) return alloc.alloc(alloc.user, bytes, device);
        void *p = nullptr;
        if (cudaMalloc(&p, bytes) != cudaSuccess) {
            cudaGetLastError();
            return nullptr;
        }
        return p;
    }
    void dev_free(void *p)
    {
        if (!p) return;
        if (alloc.free) alloc.free(alloc.user, p, device);
        else cudaFree(p);
    }
};

#define MR_CUDA(ctx, call)                                              \
    do {                                                                \
        cudaError_t e_ = (call);                                        \
        if (e_ != cudaSuccess) return (ctx)->fail_cuda(e_, #call);      \
    } while (0)

// The set-up calls free or replace buffers the producer ring's ship path (other threads) dereferences: refused while a ring is open.
#define MR_NO_RING(ctx, what) \
    if ((ctx)->ring) return (ctx)->fail(MR_ERR_STATE, std::string(what) + ": close the producer ring first (mr_ring_close)")

#define MR_ENTER(ctx)                                                                      \
    if (!(ctx)) return MR_ERR_INVALID_ARG;                                                 \
    if ((ctx)->sticky_cuda) return MR_ERR_CUDA;                                            \
    DeviceGuard guard_((ctx)->device);                                                     \
    (ctx)->err.clear()

namespace {

// LAYOUT_K4F: bring d_tally up to date (queued on the stream).  No-op unless in-record sums are pending.
cudaError_t flush_fused(mr_ctx *c)
{
    if (!c->fused || !c->fused_dirty || !c->d_recs || !c->d_tally) return cudaSuccess;
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    const unsigned grid = (unsigned)std::min<long long>((c->ncell + 255) / 256, (long long)sms * 16);
    flush_fused_kernel<<<grid, 256, 0, c->stream>>>(c->d_recs, c->d_tally, c->ncell);
    c->launches += 1;
    c->fused_dirty = false;
    return cudaGetLastError();
}

// Tile-ordered accumulators of the dictionary path: bring d_tally up to date (queued on the stream).
cudaError_t flush_tiled(mr_ctx *c)
{
    if (!c->tiled_dirty || !c->d_tally_t || !c->d_tally) return cudaSuccess;
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    const unsigned grid = (unsigned)std::min<long long>((c->ncell + 255) / 256, (long long)sms * 16);
    const int xs = c->tile_bits == 16 ? 2 : 3, ys = c->tile_bits == 4 ? 3 : 2;
    flush_tiled_kernel<<<grid, 256, 0, c->stream>>>(c->d_tally_t, c->d_tally, c->nx, c->ny, c->nz, c->ntx, c->nty, xs, ys);
    c->launches += 1;
    c->tiled_dirty = false;
    return cudaGetLastError();
}

// Everything the cast kernels accumulate outside d_tally (in-record sums, tile-ordered accumulators) -> d_tally.
cudaError_t flush_accumulators(mr_ctx *c)
{
    const cudaError_t e = flush_fused(c);
    return e != cudaSuccess ? e : flush_tiled(c);
}

void free_materials(mr_ctx *c)
{
    if (flush_accumulators(c) == cudaSuccess) cudaStreamSynchronize(c->stream);   // the sums live in buffers about to go
    c->fused = false;
    c->dev_free(c->d_tally_t);
    c->d_tally_t = nullptr;
    c->tally_t_cells = 0;
    c->tiled_dirty = false;
    c->dev_free(c->d_recs);
    c->dev_free(c->d_ids);
    c->dev_free(c->d_dict);
    c->dev_free(c->d_tiles);
    c->dev_free(c->d_crecs);
    c->d_recs = nullptr;
    c->d_ids = nullptr;
    c->d_dict = c->d_tiles = nullptr;
    c->d_crecs = nullptr;
    c->cshift = 0;
    c->ndict = 0;
    c->layout = 0;
    c->K = 0;
}

void unref_grid(mr_ctx *c, mr_ctx::Grid *g)
{
    if (!g || --g->refs > 0) return;
    c->dev_free(g->d_E);
    c->dev_free(g->d_first);
    c->grids.erase(std::remove(c->grids.begin(), c->grids.end(), g), c->grids.end());
    delete g;
}

void free_tables(mr_ctx *c)
{
    for (mr_ctx::Grid *g : c->grid_of) unref_grid(c, g);
    for (void *p : c->d_S) c->dev_free(p);
    c->grid_of.clear();
    c->d_S.clear();
    c->xs_n.clear();
    c->mix.clear();
    c->dev_free(c->d_xs);
    c->d_xs = nullptr;
    c->xs_dirty = true;
}

void free_defer(mr_ctx *c)
{
    c->dev_free(c->d_defer_cells);
    c->dev_free(c->d_defer_scores);
    c->dev_free(c->d_defer_table);
    c->dev_free(c->d_defer_ctl);
    c->d_defer_cells = nullptr;
    c->d_defer_scores = nullptr;
    c->d_defer_table = nullptr;
    c->d_defer_ctl = nullptr;
    c->defer_pool_chunks = c->defer_max_chunks = 0;
    c->defer_pending = false;
}

void free_stage(mr_ctx *c)
{
    for (int s = 0; s < kStageSlots; ++s) {
        if (c->pinned[s]) cudaFreeHost(c->pinned[s]);
        c->dev_free(c->d_stage[s]);
        c->pinned[s] = nullptr;
        c->d_stage[s] = nullptr;
    }
    c->stage_cap_rays = 0;
}

constexpr int kDictMax = 1024;   // distinct cell records the cast kernel keeps in shared memory (16 KB)

// Dictionary + tiled 2-byte index of the cell records (see mr_ctx::d_dict).  The records are formed exactly as
// pack_cells_kernel forms them (r = (float)(frac * density), empty slot = {0, id 0}), in the K = 3 encoding whatever K <= 3 is.
// Gives up (leaves ndict = 0) as soon as more than kDictMax distinct records have been seen.
int build_tiled_index(mr_ctx *c, int M, const double *density, int K, const int32_t *cell_mat, const double *cell_frac)
{
    c->ndict = 0;
    if (!c->tiled_opt || c->precision != MR_PRECISION_MIXED || K > 3 || c->mesh_rz) return MR_OK;
    struct Key {
        uint32_t w[4];
        bool operator==(const Key &o) const { return std::memcmp(w, o.w, 16) == 0; }
    };
    struct Hash {
        size_t operator()(const Key &k) const
        {
            uint64_t h = 0xcbf29ce484222325ULL;
            for (int i = 0; i < 4; ++i) h = (h ^ k.w[i]) * 0x100000001b3ULL;
            return (size_t)h;
        }
    };
    std::unordered_map<Key, uint16_t, Hash> dict;
    std::vector<Key> entries;
    std::vector<uint16_t> id_of((size_t)c->ncell);
    for (long long cell = 0; cell < c->ncell; ++cell) {
        Key k{{0u, 0u, 0u, 0u}};
        for (int s = 0; s < K; ++s) {
            const int m = cell_mat[cell * K + s];
            if (m < 0) continue;                              // empty slot: r = 0, id = 0
            const float r = (float)(cell_frac[cell * K + s] * density[m]);
            std::memcpy(&k.w[s], &r, 4);
            k.w[3] |= (uint32_t)m << (8 * s);
        }
        auto it = dict.find(k);
        if (it == dict.end()) {
            if ((int)entries.size() >= kDictMax) return MR_OK;   // too many distinct records: keep the plain layout
            it = dict.emplace(k, (uint16_t)entries.size()).first;
            entries.push_back(k);
        }
        id_of[(size_t)cell] = it->second;
    }
    // index width by dictionary size: 4 bits (tiles of 8 x 8 cells), 8 bits (8 x 4), 16 bits (4 x 4); 32 bytes per tile
    const int bits = entries.size() <= 16 ? 4 : (entries.size() <= 256 ? 8 : 16);
    const int xs = bits == 16 ? 2 : 3, ys = bits == 4 ? 3 : 2;
    const int nx = c->nx, ny = c->ny, nz = c->nz;
    const int ntx = (nx + (1 << xs) - 1) >> xs, nty = (ny + (1 << ys) - 1) >> ys;
    std::vector<uint32_t> tiles((size_t)ntx * nty * nz * 8, 0u);
    for (long long cell = 0; cell < c->ncell; ++cell) {
        const int ix = (int)(cell % nx), iy = (int)((cell / nx) % ny), iz = (int)(cell / ((long long)nx * ny));
        const size_t tile = (size_t)(ix >> xs) + (size_t)ntx * ((size_t)(iy >> ys) + (size_t)nty * iz);
        const int e = ((iy & ((1 << ys) - 1)) << xs) | (ix & ((1 << xs) - 1));
        const int bit = e * bits;
        tiles[tile * 8 + (size_t)(bit >> 5)] |= (uint32_t)id_of[(size_t)cell] << (bit & 31);
    }
    (void)M;
    uint4 *d_dict = (uint4 *)c->dev_alloc(sizeof(uint4) * kDictMax);
    uint4 *d_tiles = (uint4 *)c->dev_alloc(tiles.size() * 4);
    // tile-ordered accumulators: one double per tile entry (positions are 31-bit in the kernel)
    const long long acc_cells = ((long long)ntx * nty * nz) << (xs + ys);
    double *d_acc = acc_cells < (1LL << 31) ? (double *)c->dev_alloc((size_t)acc_cells * 8) : nullptr;
    if (!d_dict || !d_tiles || (!d_acc && acc_cells < (1LL << 31))) {
        c->dev_free(d_dict);
        c->dev_free(d_tiles);
        c->dev_free(d_acc);
        return c->fail(MR_ERR_OOM, "device allocation failed (tiled mixture index)");
    }
    cudaError_t e = cudaMemcpyAsync(d_dict, entries.data(), entries.size() * 16, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_tiles, tiles.data(), tiles.size() * 4, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess && d_acc) e = cudaMemsetAsync(d_acc, 0, (size_t)acc_cells * 8, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) {
        c->dev_free(d_dict);
        c->dev_free(d_tiles);
        c->dev_free(d_acc);
        return c->fail_cuda(e, "mr_load_materials (tiled index)");
    }
    c->d_dict = d_dict;
    c->d_tiles = d_tiles;
    c->d_tally_t = d_acc;
    c->tally_t_cells = d_acc ? acc_cells : 0;
    c->tiled_dirty = false;
    c->ndict = (int)entries.size();
    c->ntx = ntx;
    c->nty = nty;
    c->tile_bits = bits;
    return MR_OK;
}

constexpr int kCoarseMaxShift = 5;        // blocks of up to 32^3 cells
constexpr long long kCoarseMinCells = 1 << 15;

// Coarse-grid records (see mr_ctx::d_crecs).  A cell whose coordinates share exactly l low zero bits (l < kCoarseMaxShift)
// is compared with the cell whose coordinates have the low l+1 bits cleared; a difference rules out every block size
// 2^j, j > l.  If no comparison at levels 1..s fails, every aligned 2^s block holds one composition (by induction up the
// chain of those parents).  Compared are the caller's (material, fraction) slots, bit for bit.
int build_coarse_records(mr_ctx *c, const double *density, int K, const int32_t *cell_mat, const double *cell_frac)
{
    c->cshift = 0;
    if (!c->coarse_opt || c->precision != MR_PRECISION_MIXED || K > 4 || c->mesh_rz || c->ncell < kCoarseMinCells) return MR_OK;
    const int nx = c->nx, ny = c->ny, nz = c->nz;
    std::atomic<int> fail_mask{0};           // bit j: some 2^j block is not constant
    auto same = [&](long long a, long long b) {
        for (int k = 0; k < K; ++k) {
            const int ma = cell_mat[a * K + k], mb = cell_mat[b * K + k];
            if (ma != mb) return false;
            if (ma >= 0 && std::memcmp(&cell_frac[a * K + k], &cell_frac[b * K + k], 8) != 0) return false;
        }
        return true;
    };
    auto scan = [&](int z0, int z1) {
        int local = 0;
        for (int iz = z0; iz < z1; ++iz) {
            if (fail_mask.load(std::memory_order_relaxed) & 2) return;      // not even 2^3-cell blocks: give up
            for (int iy = 0; iy < ny; ++iy)
                for (int ix = 0; ix < nx; ++ix) {
                    const unsigned bits = (unsigned)(ix | iy | iz) | (1u << kCoarseMaxShift);
                    const int l = __builtin_ctz(bits);
                    if (l >= kCoarseMaxShift || (local >> (l + 1)) & 1) continue;
                    const int m = ~((2 << l) - 1);
                    const long long me = ix + (long long)nx * (iy + (long long)ny * iz);
                    const long long pa = (ix & m) + (long long)nx * ((iy & m) + (long long)ny * (iz & m));
                    if (!same(me, pa)) {
                        local |= 1 << (l + 1);
                        fail_mask.fetch_or(1 << (l + 1), std::memory_order_relaxed);
                    }
                }
        }
    };
    {
        const int T = (int)std::max(1u, std::min(16u, std::min(std::thread::hardware_concurrency(), (unsigned)nz)));
        std::vector<std::thread> pool;
        for (int t = 1; t < T; ++t) pool.emplace_back(scan, (int)((long long)nz * t / T), (int)((long long)nz * (t + 1) / T));
        scan(0, (int)((long long)nz / T));
        for (std::thread &th : pool) th.join();
    }
    int s = 0;
    while (s < kCoarseMaxShift && !((fail_mask.load() >> (s + 1)) & 1)) ++s;
    if (s == 0) return MR_OK;
    const int cnx = (nx + (1 << s) - 1) >> s, cny = (ny + (1 << s) - 1) >> s, cnz = (nz + (1 << s) - 1) >> s;
    std::vector<uint32_t> recs((size_t)cnx * cny * cnz * 8, 0u);
    for (int bz = 0; bz < cnz; ++bz)
        for (int by = 0; by < cny; ++by)
            for (int bx = 0; bx < cnx; ++bx) {
                const long long cell = ((long long)bx << s) + (long long)nx * (((long long)by << s) + (long long)ny * ((long long)bz << s));
                uint32_t *r = &recs[((size_t)bx + (size_t)cnx * ((size_t)by + (size_t)cny * bz)) * 8];
                for (int k = 0; k < K; ++k) {
                    const int m = cell_mat[cell * K + k];
                    if (m < 0) continue;                              // empty slot: r = 0, id = 0
                    const float v = (float)(cell_frac[cell * K + k] * density[m]);
                    std::memcpy(&r[k], &v, 4);
                    r[4] |= (uint32_t)m << (8 * k);
                }
            }
    void *d = c->dev_alloc(recs.size() * 4);
    if (!d) return c->fail(MR_ERR_OOM, "device allocation failed (coarse cell records)");
    cudaError_t e = cudaMemcpyAsync(d, recs.data(), recs.size() * 4, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) {
        c->dev_free(d);
        return c->fail_cuda(e, "mr_load_materials (coarse records)");
    }
    c->d_crecs = d;
    c->cshift = s;
    c->cnx = cnx;
    c->cny = cny;
    c->cnz = cnz;
    return MR_OK;
}

bool finite_increasing(const double *a, int n)
{
    for (int i = 0; i < n; ++i) {
        if (!std::isfinite(a[i])) return false;
        if (i && !(a[i] > a[i - 1])) return false;
    }
    return true;
}

template <typename K>
int set_smem(mr_ctx *c, K kernel, size_t bytes)
{
    if (bytes > 48 * 1024) MR_CUDA(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return MR_OK;
}

size_t edges_smem_bytes(const mr_ctx *c) { return sizeof(double) * (size_t)((c->nedges + 1) & ~1); }

MeshDev mesh_dev(const mr_ctx *c)
{
    MeshDev m{c->nx, c->ny, c->nz, c->nedges, c->d_edges, {c->mesh_e0[0], c->mesh_e0[1], c->mesh_e0[2]},
              {c->mesh_h[0], c->mesh_h[1], c->mesh_h[2]}};
    return m;
}

int edge_mode(const mr_ctx *c, size_t other_smem)
{
    if (c->mesh_arith) return EDGES_ARITH;
    if (edges_smem_bytes(c) <= kEdgesSmemMax && edges_smem_bytes(c) + other_smem <= 200 * 1024) return EDGES_SHARED;
    return EDGES_GLOBAL;
}

template <typename Real, typename Rec, int MODE>
int launch_cast_m(mr_ctx *c, const CastParams &P, int block, size_t smem)
{
    const long long grid = (P.n + block - 1) / block;
    if (grid > 0x7fffffffLL) return c->fail(MR_ERR_UNSUPPORTED, "batch too large for one launch");
    if (int rc = set_smem(c, cast_kernel<Real, Rec, MODE>, smem)) return rc;
    cast_kernel<Real, Rec, MODE><<<(unsigned)grid, block, smem, c->work_stream()>>>(P);
    c->launches += 1;
    MR_CUDA(c, cudaGetLastError());
    return MR_OK;
}

template <typename Real, typename Rec>
int launch_cast_t(mr_ctx *c, const CastParams &P)
{
    const int block = c->block_threads;
    const size_t per_block = walker_smem_bytes(block) + (size_t)(c->M + c->N) * block * sizeof(Real) +
                             (rec_per_entry<Rec>::value ? (size_t)kPerEntryMax * block * sizeof(Real) : 0) +
                             (Rec::kTiled ? (size_t)c->ndict * sizeof(uint4) : 0);
    const int mode = edge_mode(c, per_block);
    const size_t smem = (mode == EDGES_SHARED ? edges_smem_bytes(c) : 0) + per_block;
    if (smem > 227 * 1024) return c->fail(MR_ERR_UNSUPPORTED, "materials x block threads exceed shared memory; lower MR_OPT_BLOCK_THREADS");
    switch (mode) {
    case EDGES_ARITH: return launch_cast_m<Real, Rec, EDGES_ARITH>(c, P, block, smem);
    case EDGES_SHARED: return launch_cast_m<Real, Rec, EDGES_SHARED>(c, P, block, smem);
    default: return launch_cast_m<Real, Rec, EDGES_GLOBAL>(c, P, block, smem);
    }
}

template <typename Real, typename Rec, int MODE>
int launch_coop_m(mr_ctx *c, const CastParams &P, int block, size_t smem)
{
    const long long grid = (P.n + block - 1) / block;
    if (grid > 0x7fffffffLL) return c->fail(MR_ERR_UNSUPPORTED, "batch too large for one launch");
    if (c->coop_opt == 3) {     // pair exchange by shuffles instead of the 8-step staging
        if (int rc = set_smem(c, cast_coop_kernel<Real, Rec, MODE, true>, smem)) return rc;
        cast_coop_kernel<Real, Rec, MODE, true><<<(unsigned)grid, block, smem, c->work_stream()>>>(P);
        c->launches += 1;
        MR_CUDA(c, cudaGetLastError());
        return MR_OK;
    }
    if (int rc = set_smem(c, cast_coop_kernel<Real, Rec, MODE>, smem)) return rc;
    cast_coop_kernel<Real, Rec, MODE><<<(unsigned)grid, block, smem, c->work_stream()>>>(P);
    c->launches += 1;
    MR_CUDA(c, cudaGetLastError());
    return MR_OK;
}

// cast_coop_kernel (cooperative, transposed tally adds) for the record types it is built for
template <typename Real, typename Rec>
int launch_coop_t(mr_ctx *c, const CastParams &P)
{
    const int block = c->block_threads;
    const size_t per_block = walker_smem_bytes(block) + (((size_t)(c->M + c->N) * block * sizeof(Real) + 15) & ~(size_t)15) +
                             (rec_per_entry<Rec>::value ? (size_t)kPerEntryMax * block * sizeof(Real) : 0) +
                             (Rec::kTiled ? (size_t)c->ndict * sizeof(uint4) : 0) + (size_t)(block / 32) * coop_warp_smem_bytes();
    const int mode = edge_mode(c, per_block);
    const size_t smem = (mode == EDGES_SHARED ? edges_smem_bytes(c) : 0) + per_block;
    if (smem > 227 * 1024) return launch_cast_t<Real, Rec>(c, P);
    switch (mode) {
    case EDGES_ARITH: return launch_coop_m<Real, Rec, EDGES_ARITH>(c, P, block, smem);
    case EDGES_SHARED: return launch_coop_m<Real, Rec, EDGES_SHARED>(c, P, block, smem);
    default: return launch_coop_m<Real, Rec, EDGES_GLOBAL>(c, P, block, smem);
    }
}

template <typename Real, typename Rec>
int launch_cast_or_coop(mr_ctx *c, const CastParams &P, bool coop_auto_always = false)
{
    // auto: contended, L2-resident tallies -- and the 16-byte record-pair path at any size, where a segment costs an L2 request
    // for its record as well as for its add (config 3 with the dictionary off: 8.42 -> 7.80 ms)
    const bool coop = c->coop_opt == 1 || c->coop_opt == 3 ||
                      (c->coop_opt == 2 && (coop_auto_always || c->resident_bytes() <= c->l2_bytes / 2));
    return coop ? launch_coop_t<Real, Rec>(c, P) : launch_cast_t<Real, Rec>(c, P);
}

// cast_tiled_kernel (mr_tiled.cuh): the dictionary path with tile-ordered accumulators
template <int BITS, int MODE, bool COOP>
int launch_tiled_m(mr_ctx *c, const CastParams &P, int block, size_t smem)
{
    const long long grid = (P.n + block - 1) / block;
    if (grid > 0x7fffffffLL) return c->fail(MR_ERR_UNSUPPORTED, "batch too large for one launch");
    if (int rc = set_smem(c, cast_tiled_kernel<BITS, MODE, COOP>, smem)) return rc;
    cast_tiled_kernel<BITS, MODE, COOP><<<(unsigned)grid, block, smem, c->work_stream()>>>(P);
    c->launches += 1;
    MR_CUDA(c, cudaGetLastError());
    return MR_OK;
}

template <int BITS, bool COOP>
int launch_tiled_c(mr_ctx *c, const CastParams &P)
{
    const int block = c->block_threads;
    const size_t per_block = walker_smem_bytes(block) + (((size_t)(c->M + c->N) * block * sizeof(float) + 15) & ~(size_t)15) +
                             (BITS == 4 ? (size_t)kPerEntryMax * block * sizeof(float) : 0) + (size_t)c->ndict * sizeof(uint4) +
                             (COOP ? (size_t)(block / 32) * coop_warp_smem_bytes() : 0);
    const int mode = edge_mode(c, per_block);
    const size_t smem = (mode == EDGES_SHARED ? edges_smem_bytes(c) : 0) + per_block;
    if (smem > 227 * 1024) return c->fail(MR_ERR_UNSUPPORTED, "materials x block threads exceed shared memory; lower MR_OPT_BLOCK_THREADS");
    switch (mode) {
    case EDGES_ARITH: return launch_tiled_m<BITS, EDGES_ARITH, COOP>(c, P, block, smem);
    case EDGES_SHARED: return launch_tiled_m<BITS, EDGES_SHARED, COOP>(c, P, block, smem);
    default: return launch_tiled_m<BITS, EDGES_GLOBAL, COOP>(c, P, block, smem);
    }
}

bool use_coop(const mr_ctx *c) { return c->coop_opt == 1 || (c->coop_opt == 2 && c->resident_bytes() <= c->l2_bytes / 2); }

template <int BITS>
int launch_tiled(mr_ctx *c, const CastParams &P)
{
    c->tiled_dirty = true;
    return use_coop(c) ? launch_tiled_c<BITS, true>(c, P) : launch_tiled_c<BITS, false>(c, P);
}

int upload_xs_desc(mr_ctx *c)
{
    if (!c->xs_dirty) return MR_OK;
    // descriptors: [0, M) materials (n = 0: a nuclide mixture), [M, M + N) nuclides (n = 0: not loaded)
    int N = 0;
    for (int q = 0; q < MR_MAX_NUCLIDES; ++q)
        if (c->nuc_n[q] > 0) N = q + 1;
    bool any_mix = false;
    for (int m = 0; m < c->M; ++m) any_mix = any_mix || !c->mix[m].empty();
    if (!any_mix) N = 0;
    std::vector<XsDesc> h(c->M + N);
    for (int m = 0; m < c->M; ++m) {
        const mr_ctx::Grid *g = c->grid_of[m];
        h[m] = g ? XsDesc{g->d_E, c->d_S[m], c->xs_n[m], g->id, g->d_first, g->b0, g->sh} : XsDesc{nullptr, nullptr, 0, -1, nullptr, 0, 0};
    }
    for (int q = 0; q < N; ++q) {
        const mr_ctx::Grid *g = c->nuc_grid_of[q];
        h[c->M + q] = g ? XsDesc{g->d_E, c->nuc_S[q], c->nuc_n[q], g->id, g->d_first, g->b0, g->sh} : XsDesc{nullptr, nullptr, 0, -1, nullptr, 0, 0};
    }
    if (!c->d_xs) {
        c->d_xs = (XsDesc *)c->dev_alloc(sizeof(XsDesc) * (MR_MAX_MATERIALS + MR_MAX_NUCLIDES));
        if (!c->d_xs) return c->fail(MR_ERR_OOM, "device allocation failed (table descriptors)");
    }
    MR_CUDA(c, cudaMemcpyAsync(c->d_xs, h.data(), sizeof(XsDesc) * h.size(), cudaMemcpyHostToDevice, c->stream));
    // mixtures: offsets per material, then (nuclide, weight) entries; weights rounded once to fp32 in MIXED mode
    std::vector<int> off(c->M + 1, 0), nuc;
    std::vector<double> wd;
    std::vector<float> wf;
    for (int m = 0; m < c->M; ++m) {
        for (const auto &e : c->mix[m]) {
            nuc.push_back(e.first);
            wd.push_back(e.second);
            wf.push_back((float)e.second);
        }
        off[m + 1] = (int)nuc.size();
    }
    if (N > 0) {
        if (!c->d_mix_off) {
            c->d_mix_off = (int *)c->dev_alloc(sizeof(int) * (MR_MAX_MATERIALS + 1));
            c->d_mix_nuc = (int *)c->dev_alloc(sizeof(int) * MR_MAX_MATERIALS * MR_MAX_MIX);
            c->d_mix_w = c->dev_alloc(sizeof(double) * MR_MAX_MATERIALS * MR_MAX_MIX);
            if (!c->d_mix_off || !c->d_mix_nuc || !c->d_mix_w) return c->fail(MR_ERR_OOM, "device allocation failed (mixtures)");
        }
        const bool dbl = c->precision == MR_PRECISION_DOUBLE;
        MR_CUDA(c, cudaMemcpyAsync(c->d_mix_off, off.data(), sizeof(int) * off.size(), cudaMemcpyHostToDevice, c->stream));
        MR_CUDA(c, cudaMemcpyAsync(c->d_mix_nuc, nuc.data(), sizeof(int) * nuc.size(), cudaMemcpyHostToDevice, c->stream));
        MR_CUDA(c, cudaMemcpyAsync(c->d_mix_w, dbl ? (const void *)wd.data() : (const void *)wf.data(),
                                   (dbl ? sizeof(double) : sizeof(float)) * nuc.size(), cudaMemcpyHostToDevice, c->stream));
    }
    MR_CUDA(c, cudaStreamSynchronize(c->stream));  // the host vectors go out of scope
    c->N = N;
    c->xs_dirty = false;
    return MR_OK;
}

int ready_to_cast(mr_ctx *c)
{
    if (!c->d_tally) return c->fail(MR_ERR_STATE, "no mesh loaded");
    if (!c->d_recs) return c->fail(MR_ERR_STATE, "no materials loaded");
    for (int m = 0; m < c->M; ++m) {
        if (m < (int)c->xs_n.size() && c->xs_n[m] > 0) continue;
        if (m >= (int)c->mix.size() || c->mix[m].empty())
            return c->fail(MR_ERR_STATE, "cross-section table of material " + std::to_string(m) + " not loaded");
        for (const auto &e : c->mix[m])
            if (c->nuc_n[e.first] == 0)
                return c->fail(MR_ERR_STATE, "material " + std::to_string(m) + " needs nuclide " + std::to_string(e.first) + ", whose table is not loaded");
    }
    return MR_OK;
}

constexpr long long kSortMinRays = 1 << 14;   // below this a batch is a handful of CTAs: ordering buys nothing

// Queue the ordering pre-pass for n device-resident rays; *perm_out = null if the batch is cast in buffer order.
// nsec > 0: next-event mode, one section per detector det_first .. det_first + nsec - 1 (keys, perm: n entries per
// section; histogram: nkeys + 1 entries per section).
int order_rays(mr_ctx *c, long long n, const void *d_rays, const uint32_t **perm_out, int nsec = 0, int det_first = 0)
{
    *perm_out = nullptr;
    const int L = c->lane;
    cudaStream_t ws = c->work_stream();
    uint32_t *&d_keys = c->d_keys_l[L], *&d_perm = c->d_perm_l[L], *&d_hist = c->d_hist_l[L], *&d_blk_hist = c->d_blk_hist_l[L];
    long long &sort_cap = c->sort_cap_l[L], &hist_cap = c->hist_cap_l[L], &blk_hist_cap = c->blk_hist_cap_l[L];
    if (!c->sort_rays || c->mesh_rz || n < kSortMinRays || n > 0xffffffffLL || edges_smem_bytes(c) > kEdgesSmemMax) return MR_OK;
    const int sections = std::max(nsec, 1);
    const int nlen = 128;
    const int zdiv = (c->nz + 255) / 256;
    const int nslab = (c->nz + zdiv - 1) / zdiv;
    const int maxlen = c->nx + c->ny + c->nz;
    int lshift = 0;
    while ((maxlen >> lshift) >= nlen) ++lshift;
    const int nkeys = nslab * nlen + 1;
    const long long entries = n * sections;
    if (entries > sort_cap) {
        MR_CUDA(c, cudaStreamSynchronize(ws));
        c->dev_free(d_keys);
        c->dev_free(d_perm);
        d_keys = (uint32_t *)c->dev_alloc((size_t)entries * 4);
        d_perm = (uint32_t *)c->dev_alloc((size_t)entries * 4);
        sort_cap = (d_keys && d_perm) ? entries : 0;
        if (!sort_cap) {
            c->dev_free(d_keys);
            c->dev_free(d_perm);
            d_keys = d_perm = nullptr;
            return c->fail(MR_ERR_OOM, "device allocation failed (ray ordering scratch)");
        }
    }
    const long long hist_entries = (long long)(nkeys + 1) * sections;
    if (hist_entries > hist_cap) {
        MR_CUDA(c, cudaStreamSynchronize(ws));
        c->dev_free(d_hist);
        d_hist = (uint32_t *)c->dev_alloc((size_t)hist_entries * 4);
        hist_cap = d_hist ? hist_entries : 0;
        if (!d_hist) return c->fail(MR_ERR_OOM, "device allocation failed (ray ordering histogram)");
    }
    SortParams S{mesh_dev(c), d_rays, n, c->precision == MR_PRECISION_DOUBLE ? 1 : 0,
                 zdiv, lshift, nlen, nkeys, d_keys, d_hist, d_perm, nsec > 0 ? c->d_det : nullptr, det_first,
                 c->order_mode == 2 || (c->order_mode == 0 && (c->resident_bytes() <= c->l2_bytes / 2 || c->order_longest_auto)) ? 1 : 0, nslab,
                 c->mesh_arith ? 1 : 0, 0, nullptr};
    const size_t smem = edges_smem_bytes(c);
    // Block-local variant: every CTA counts its own contiguous share of the rays in shared memory, so neither pass
    // needs a global atomic.  Used when the counters fit beside the plane table; else the global-atomic kernels.
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    const size_t cnt_smem = smem + (size_t)nkeys * 4;
    const int nblk = (int)std::max<long long>(1, std::min<long long>(sms, n / 4096));
    if (cnt_smem <= 200 * 1024) {
        const long long need = (long long)sections * nblk * nkeys;
        if (need > blk_hist_cap) {
            MR_CUDA(c, cudaStreamSynchronize(ws));
            c->dev_free(d_blk_hist);
            d_blk_hist = (uint32_t *)c->dev_alloc((size_t)need * 4);
            blk_hist_cap = d_blk_hist ? need : 0;
            if (!d_blk_hist) return c->fail(MR_ERR_OOM, "device allocation failed (ray ordering block histograms)");
        }
        S.nblk = nblk;
        S.blk_hist = d_blk_hist;
        const dim3 gblk((unsigned)nblk, (unsigned)sections), gkey((unsigned)((nkeys + 255) / 256), (unsigned)sections);
        if (int rc = set_smem(c, count_kernel, cnt_smem)) return rc;
        if (int rc = set_smem(c, place_kernel, (size_t)nkeys * 4)) return rc;
        count_kernel<<<gblk, 1024, cnt_smem, ws>>>(S);
        key_totals_kernel<<<gkey, 256, 0, ws>>>(S);
        scan_kernel<<<sections, 1024, 0, ws>>>(d_hist, nkeys);
        block_offsets_kernel<<<gkey, 256, 0, ws>>>(S);
        place_kernel<<<gblk, 1024, (size_t)nkeys * 4, ws>>>(S);
        c->launches += 5;
    } else {
        MR_CUDA(c, cudaMemsetAsync(d_hist, 0, (size_t)hist_entries * 4, ws));
        const dim3 grid((unsigned)((n + 255) / 256), (unsigned)sections);
        if (int rc = set_smem(c, classify_kernel, smem)) return rc;
        classify_kernel<<<grid, 256, smem, ws>>>(S);
        scan_kernel<<<sections, 1024, 0, ws>>>(d_hist, nkeys);
        scatter_kernel<<<grid, 256, 0, ws>>>(S);
        c->launches += 3;
    }
    MR_CUDA(c, cudaGetLastError());
    *perm_out = d_perm;
    return MR_OK;
}

template <typename Real, typename Rec, bool TRACE>
int launch_rz_t(mr_ctx *c, const RzParams &Q, int block)
{
    const size_t smem = edges_smem_bytes(c) + rz_re2_bytes(c->nx) + (TRACE ? 0 : (((size_t)(c->M + c->N) * block * sizeof(Real) + 15) & ~(size_t)15) +
                                                           (size_t)(block / 32) * coop_warp_smem_bytes());
    if (smem > 227 * 1024) return c->fail(MR_ERR_UNSUPPORTED, "rz mesh: planes and materials exceed shared memory");
    if (int rc = set_smem(c, rz_kernel<Real, Rec, TRACE>, smem)) return rc;
    // persistent kernel: as many CTAs as can be resident; lanes pull rays from counters[3]
    int sms = 148, per_sm = 1;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    MR_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, rz_kernel<Real, Rec, TRACE>, block, smem));
    const long long grid = std::max<long long>(1, std::min<long long>((Q.c.n + block - 1) / block, (long long)sms * std::max(per_sm, 1)));
    MR_CUDA(c, cudaMemsetAsync(c->d_counters + 3, 0, sizeof(unsigned long long), c->work_stream()));
    rz_kernel<Real, Rec, TRACE><<<(unsigned)grid, block, smem, c->work_stream()>>>(Q);
    c->launches += 1;
    MR_CUDA(c, cudaGetLastError());
    return MR_OK;
}

int launch_rz_cast(mr_ctx *c, const CastParams &P)
{
    RzParams Q{};
    Q.c = P;
    Q.spherical = c->mesh_sphere ? 1 : 0;
    // every CTA stages the radii and planes in shared memory: 256 threads amortise that table over twice the warps
    const int block = c->rz_block_threads;
    if (c->precision == MR_PRECISION_DOUBLE)
        return c->layout == LAYOUT_DK3 ? launch_rz_t<double, CellRec<LAYOUT_DK3>, false>(c, Q, block)
                                       : launch_rz_t<double, CellRecGeneric<double>, false>(c, Q, block);
    switch (c->layout) {
    case LAYOUT_K1: return launch_rz_t<float, QuadRecK1, false>(c, Q, block);
    case LAYOUT_K2: return launch_rz_t<float, CellRec<LAYOUT_K2P>, false>(c, Q, block);
    case LAYOUT_K3: return launch_rz_t<float, CellRec<LAYOUT_K3P>, false>(c, Q, block);
    case LAYOUT_K4: return launch_rz_t<float, CellRec<LAYOUT_K4>, false>(c, Q, block);
    case LAYOUT_D8: return launch_rz_t<float, CellRec<LAYOUT_D8>, false>(c, Q, block);
    default: return launch_rz_t<float, CellRecGeneric<float>, false>(c, Q, block);
    }
}

template <typename Real, typename Rec, bool TRACE>
int launch_rz_ne_t(mr_ctx *c, const RzNextEventParams &Q, int block)
{
    const size_t smem = edges_smem_bytes(c) + (size_t)(c->M + c->N) * block * sizeof(Real);
    if (smem > 227 * 1024) return c->fail(MR_ERR_UNSUPPORTED, "rz mesh: planes and materials exceed shared memory");
    if (int rc = set_smem(c, rz_next_event_kernel<Real, Rec, TRACE>, smem)) return rc;
    int sms = 148, per_sm = 1;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    MR_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, rz_next_event_kernel<Real, Rec, TRACE>, block, smem));
    const long long pairs = Q.c.n * Q.ndet;
    const long long grid = std::max<long long>(1, std::min<long long>((pairs + block - 1) / block, (long long)sms * std::max(per_sm, 1)));
    MR_CUDA(c, cudaMemsetAsync(Q.work, 0, sizeof(unsigned long long), c->work_stream()));
    rz_next_event_kernel<Real, Rec, TRACE><<<(unsigned)grid, block, smem, c->work_stream()>>>(Q);
    c->launches += 1;
    MR_CUDA(c, cudaGetLastError());
    return MR_OK;
}

// next-event cast on an R-Z / spherical mesh: n device-resident events against detectors det_first .. det_first + ndet - 1
template <bool TRACE>
int launch_rz_next_event(mr_ctx *c, RzNextEventParams Q)
{
    Q.spherical = c->mesh_sphere ? 1 : 0;
    Q.work = c->d_counters + 3;
    const int block = c->block_threads;
    if (c->precision == MR_PRECISION_DOUBLE)
        return c->layout == LAYOUT_DK3 ? launch_rz_ne_t<double, CellRec<LAYOUT_DK3>, TRACE>(c, Q, block)
                                       : launch_rz_ne_t<double, CellRecGeneric<double>, TRACE>(c, Q, block);
    switch (c->layout) {
    case LAYOUT_K1: return launch_rz_ne_t<float, CellRec<LAYOUT_K1>, TRACE>(c, Q, block);
    case LAYOUT_K2: return launch_rz_ne_t<float, CellRec<LAYOUT_K2>, TRACE>(c, Q, block);
    case LAYOUT_K3: return launch_rz_ne_t<float, CellRec<LAYOUT_K3>, TRACE>(c, Q, block);
    case LAYOUT_K4: return launch_rz_ne_t<float, CellRec<LAYOUT_K4>, TRACE>(c, Q, block);
    case LAYOUT_D8: return launch_rz_ne_t<float, CellRec<LAYOUT_D8>, TRACE>(c, Q, block);
    default: return launch_rz_ne_t<float, CellRecGeneric<float>, TRACE>(c, Q, block);
    }
}

// ---- deferred tally (mr_defer.cuh) ----------------------------------------------------------------
constexpr int kDeferCtlWords = 72;

bool use_deferred(const mr_ctx *c, int path)
{
    if (c->precision != MR_PRECISION_MIXED || c->mesh_rz) return false;
    if (path != MR_PATH_COARSE && path != MR_PATH_K4) return false;
    if (c->defer_opt == 1) return true;
    return c->defer_opt == 2 && path == MR_PATH_COARSE && (size_t)c->ncell * 8 > 2 * c->l2_bytes;
}

// region size: at most an eighth of the L2 of tally per bin, at most kDeferBins bins
void defer_geometry(const mr_ctx *c, int *shift, int *nbin)
{
    int s = 10;
    while (((size_t)8 << (s + 1)) <= std::max<size_t>(c->l2_bytes / 8, (size_t)1 << 13)) ++s;
    if (c->defer_shift_fixed > 0) s = c->defer_shift_fixed;
    while (((c->ncell + (1LL << s) - 1) >> s) > kDeferBins) ++s;
    *shift = s;
    *nbin = (int)((c->ncell + (1LL << s) - 1) >> s);
}

// (Re)allocates the pool for `entries` (cell, score) pairs.  The stream must be idle.
int ensure_defer_pool(mr_ctx *c, long long entries)
{
    const long long max_chunks_total = (1LL << 20) - 1;                       // pool indices are 32-bit
    int shift, nbin;
    defer_geometry(c, &shift, &nbin);
    long long chunks = (entries + kDeferChunk - 1) / kDeferChunk;
    if (c->defer_pool_fixed == 0) {
        // every resident warp may hold one partly filled range per bin (padded when the warp drains)
        int sms = 148;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
        chunks += ((long long)sms * 32 * nbin * kDeferRange + kDeferChunk - 1) / kDeferChunk + nbin;
    }
    chunks = std::max<long long>(1, std::min(max_chunks_total, chunks));
    if (c->defer_pool_fixed == 0 ? chunks <= c->defer_pool_chunks : (chunks == c->defer_pool_chunks && c->d_defer_table)) return MR_OK;
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    if (c->stream2) MR_CUDA(c, cudaStreamSynchronize(c->stream2));
    free_defer(c);
    if (!c->h_defer_ctl) {
        MR_CUDA(c, cudaMallocHost((void **)&c->h_defer_ctl, 4 * sizeof(unsigned long long)));
        std::memset(c->h_defer_ctl, 0, 4 * sizeof(unsigned long long));
        MR_CUDA(c, cudaEventCreateWithFlags(&c->ev_defer, cudaEventDisableTiming));
    }
    const long long per_bin = std::min(chunks, 4 * chunks / std::max(nbin, 1) + 64);   // a bin may hold 4x its share
    c->d_defer_cells = (uint32_t *)c->dev_alloc((size_t)chunks * kDeferChunk * 4);
    c->d_defer_scores = (double *)c->dev_alloc((size_t)chunks * kDeferChunk * 8);
    c->d_defer_table = (int *)c->dev_alloc((size_t)nbin * per_bin * 4);
    c->d_defer_ctl = (unsigned long long *)c->dev_alloc(kDeferCtlWords * 8);
    if (!c->d_defer_cells || !c->d_defer_scores || !c->d_defer_table || !c->d_defer_ctl) {
        free_defer(c);
        return c->fail(MR_ERR_OOM, "device allocation failed (deferred-tally pool)");
    }
    MR_CUDA(c, cudaMemsetAsync(c->d_defer_ctl, 0, kDeferCtlWords * 8, c->stream));
    c->defer_pool_chunks = (int)chunks;
    c->defer_max_chunks = (int)per_bin;
    c->defer_direct_seen = 0;
    return MR_OK;
}

template <typename Rec, int MODE>
int launch_defer_m(mr_ctx *c, const CastParams &P, const DeferParams &D, size_t smem)
{
    const int block = 128;
    if (int rc = set_smem(c, cast_defer_kernel<Rec, MODE>, smem)) return rc;
    int sms = 148, per_sm = 1;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    MR_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, cast_defer_kernel<Rec, MODE>, block, smem));
    const long long grid = std::max<long long>(1, std::min<long long>((P.n + block - 1) / block, (long long)sms * std::max(per_sm, 1)));
    cast_defer_kernel<Rec, MODE><<<(unsigned)grid, block, smem, c->work_stream()>>>(P, D);
    c->launches += 1;
    MR_CUDA(c, cudaGetLastError());
    return MR_OK;
}

// The cast of P.n rays with the deferred tally: phase A (walk + score, pairs binned by tally region), phase B (bin
// after bin into the tally), in sub-batches sized to the pool.
template <typename Rec>
int cast_deferred(mr_ctx *c, CastParams P)
{
    cudaStream_t ws = c->work_stream();
    // did the previous deferred cast run out of pool?  (looked at without waiting)
    if (c->defer_pending && cudaEventQuery(c->ev_defer) == cudaSuccess) {
        c->defer_pending = false;
        if (c->h_defer_ctl[2] > c->defer_direct_seen) {
            c->defer_direct_seen = c->h_defer_ctl[2];
            c->defer_entries_per_ray *= 1.5;
        }
    } else
        cudaGetLastError();
    if (c->defer_entries_per_ray <= 0.0) c->defer_entries_per_ray = (double)(c->nx + c->ny + c->nz) / 3.0 + 8.0;
    const long long pool_cap_entries = (long long)((24ULL << 30) / 12);
    const long long want = c->defer_pool_fixed > 0 ? c->defer_pool_fixed
                         : std::max<long long>(1 << 20, std::min<long long>(pool_cap_entries, (long long)((double)P.n * c->defer_entries_per_ray)));
    if (int rc = ensure_defer_pool(c, want)) return rc;
    const long long pool_entries = std::max<long long>(kDeferChunk, std::min<long long>(want, (long long)c->defer_pool_chunks * kDeferChunk));
    const long long sub = std::max<long long>(1024, (long long)((double)pool_entries / c->defer_entries_per_ray));

    DeferParams D{};
    defer_geometry(c, &D.bin_shift, &D.nbin);
    D.max_chunks = c->defer_max_chunks;
    D.pool_chunks = c->defer_pool_chunks;
    D.cells = c->d_defer_cells;
    D.scores = c->d_defer_scores;
    D.table = c->d_defer_table;
    D.cursor = c->d_defer_ctl;
    D.pool_next = reinterpret_cast<unsigned int *>(c->d_defer_ctl + 64);
    D.work = c->d_defer_ctl + 65;
    D.direct = c->d_defer_ctl + 66;
    D.queue = reinterpret_cast<unsigned int *>(c->d_defer_ctl + 67);

    const int block = 128;
    const size_t per_block = walker_smem_bytes(block) + (((size_t)(c->M + c->N) * block * sizeof(float) + 15) & ~(size_t)15) +
                             (size_t)(block / 32) * defer_warp_smem_bytes(D.nbin);
    const int mode = edge_mode(c, per_block);
    const size_t smem = (mode == EDGES_SHARED ? edges_smem_bytes(c) : 0) + per_block;
    if (smem > 227 * 1024) return c->fail(MR_ERR_UNSUPPORTED, "deferred tally: materials and bins exceed shared memory");
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    const long long n_all = P.n;
    const char *rays0 = (const char *)P.rays;
    const uint32_t *perm0 = P.perm;
    for (long long first = 0; first < n_all; first += sub) {
        P.n = std::min(sub, n_all - first);
        if (perm0) P.perm = perm0 + first;
        else P.rays = rays0 + (size_t)first * c->ray_bytes();
        MR_CUDA(c, cudaMemsetAsync(c->d_defer_ctl, 0, 66 * 8, ws));
        MR_CUDA(c, cudaMemsetAsync(c->d_defer_ctl + 67, 0, 8, ws));
        MR_CUDA(c, cudaMemsetAsync(c->d_defer_table, 0xff, (size_t)D.nbin * D.max_chunks * 4, ws));
        int rc;
        switch (mode) {
        case EDGES_ARITH: rc = launch_defer_m<Rec, EDGES_ARITH>(c, P, D, smem); break;
        case EDGES_SHARED: rc = launch_defer_m<Rec, EDGES_SHARED>(c, P, D, smem); break;
        default: rc = launch_defer_m<Rec, EDGES_GLOBAL>(c, P, D, smem);
        }
        if (rc) return rc;
        defer_scatter_kernel<<<(unsigned)(sms * 8), 256, 0, ws>>>(D, c->d_tally);
        c->launches += 1;
        MR_CUDA(c, cudaGetLastError());
    }
    if (!c->defer_pending && !c->ring) {     // (a producer ring ships from other threads: leave the feedback to the next plain call)
        MR_CUDA(c, cudaMemcpyAsync(c->h_defer_ctl, c->d_defer_ctl + 64, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, ws));
        MR_CUDA(c, cudaEventRecord(c->ev_defer, ws));
        c->defer_pending = true;
    }
    return MR_OK;
}

// Which cell-record path mr_cast_rays takes for the resident problem (MR_INFO_RECORD_PATH).
int record_path(const mr_ctx *c)
{
    if (!c->d_recs) return MR_PATH_NONE;
    if (c->mesh_rz) return MR_PATH_RZ;
    if (c->precision == MR_PRECISION_DOUBLE) return c->layout == LAYOUT_DK3 ? MR_PATH_DOUBLE_K3 : MR_PATH_DOUBLE_GENERIC;
    if (c->ndict > 0 && c->tiled_opt && c->layout >= LAYOUT_K1 && c->layout <= LAYOUT_K3)
        return c->tile_bits == 4 ? MR_PATH_TILED4 : (c->tile_bits == 8 ? MR_PATH_TILED8 : MR_PATH_TILED16);
    if (c->cshift > 0 && c->coarse_opt && c->layout >= LAYOUT_K1 && c->layout <= LAYOUT_K4) return MR_PATH_COARSE;
    switch (c->layout) {
    case LAYOUT_K1: return MR_PATH_K1;
    case LAYOUT_K2: return c->pair_records ? MR_PATH_K2_PAIRS : MR_PATH_K2;
    case LAYOUT_K3: return c->pair_records ? MR_PATH_K3_PAIRS : MR_PATH_K3;
    case LAYOUT_K4: return (c->fused && c->defer_opt != 1 && !c->tally_borrowed) ? MR_PATH_K4_FUSED : MR_PATH_K4;
    case LAYOUT_D8: return MR_PATH_DENSE8;
    default: return MR_PATH_GENERIC;
    }
}

// Queue the cast of n device-resident rays on the context's stream.
int cast_device(mr_ctx *c, long long n, const void *d_rays)
{
    CastParams P{};
    P.mesh = mesh_dev(c);
    P.recs = c->d_recs;
    P.ids = c->d_ids;
    P.K = c->K;
    P.M = c->M;
    P.xs = c->d_xs;
    P.N = c->N;
    P.mix_off = c->d_mix_off;
    P.mix_nuc = c->d_mix_nuc;
    P.mix_w = c->d_mix_w;
    P.rays = d_rays;
    c->order_longest_auto = use_deferred(c, record_path(c));
    const int rc_order = order_rays(c, n, d_rays, &P.perm);
    c->order_longest_auto = false;
    if (rc_order) return rc_order;
    P.n = n;
    P.agg_first = c->agg_first;
    P.tally = c->d_tally;
    P.counters = c->d_counters;
    if (c->kev_used + 2 > c->kev.size()) {
        cudaEvent_t a = nullptr, b = nullptr;
        MR_CUDA(c, cudaEventCreate(&a));
        MR_CUDA(c, cudaEventCreate(&b));
        c->kev.push_back(a);
        c->kev.push_back(b);
    }
    MR_CUDA(c, cudaEventRecord(c->kev[c->kev_used], c->work_stream()));
    int rc;
    switch (record_path(c)) {
    case MR_PATH_RZ: rc = launch_rz_cast(c, P); break;
    case MR_PATH_DOUBLE_K3: rc = launch_cast_or_coop<double, CellRec<LAYOUT_DK3>>(c, P, true); break;
    case MR_PATH_DOUBLE_GENERIC: rc = launch_cast_t<double, CellRecGeneric<double>>(c, P); break;
    case MR_PATH_TILED4: case MR_PATH_TILED8: case MR_PATH_TILED16:
        P.dict = c->d_dict;
        P.tiles = c->d_tiles;
        P.ndict = c->ndict;
        P.ntx = c->ntx;
        P.nty = c->nty;
        if (c->tiled_tally_opt && c->d_tally_t && !c->tally_borrowed) {
            P.tally_t = c->d_tally_t;
            rc = c->tile_bits == 4 ? launch_tiled<4>(c, P) : c->tile_bits == 8 ? launch_tiled<8>(c, P) : launch_tiled<16>(c, P);
        } else
            rc = c->tile_bits == 4 ? launch_cast_or_coop<float, TiledRec<4>>(c, P)
               : c->tile_bits == 8 ? launch_cast_or_coop<float, TiledRec<8>>(c, P) : launch_cast_or_coop<float, TiledRec<16>>(c, P);
        break;
    case MR_PATH_COARSE:
        P.crecs = c->d_crecs;
        P.cshift = c->cshift;
        P.cnx = c->cnx;
        P.cny = c->cny;
        rc = use_deferred(c, MR_PATH_COARSE) ? cast_deferred<CellRec<LAYOUT_C4>>(c, P) : launch_cast_t<float, CellRec<LAYOUT_C4>>(c, P);
        break;
    case MR_PATH_K1: rc = launch_cast_or_coop<float, CellRec<LAYOUT_K1>>(c, P); break;
    case MR_PATH_K2: rc = launch_cast_t<float, CellRec<LAYOUT_K2>>(c, P); break;
    case MR_PATH_K3: rc = launch_cast_t<float, CellRec<LAYOUT_K3>>(c, P); break;
    case MR_PATH_K2_PAIRS: rc = launch_cast_t<float, CellRec<LAYOUT_K2P>>(c, P); break;
    case MR_PATH_K3_PAIRS: rc = launch_cast_or_coop<float, CellRec<LAYOUT_K3P>>(c, P, true); break;
    case MR_PATH_K4_FUSED: rc = launch_cast_t<float, CellRec<LAYOUT_K4F>>(c, P); c->fused_dirty = true; break;
    case MR_PATH_K4:
        rc = use_deferred(c, MR_PATH_K4) ? cast_deferred<CellRec<LAYOUT_K4>>(c, P) : launch_cast_t<float, CellRec<LAYOUT_K4>>(c, P);
        break;
    case MR_PATH_DENSE8: rc = launch_cast_or_coop<float, CellRec<LAYOUT_D8>>(c, P); break;
    default: rc = launch_cast_t<float, CellRecGeneric<float>>(c, P);
    }
    if (rc) return rc;
    MR_CUDA(c, cudaEventRecord(c->kev[c->kev_used + 1], c->work_stream()));
    c->kev_used += 2;
    return MR_OK;
}

// parallel host copy into a pinned staging slot (a single memcpy thread moves ~10 GB/s, less than the PCIe link)
void host_copy(void *dst, const void *src, size_t bytes, int threads)
{
    const size_t kMinPerThread = 4u << 20;
    int t = (int)std::min<size_t>((size_t)std::max(1, threads), bytes / kMinPerThread);
    if (t <= 1) {
        std::memcpy(dst, src, bytes);
        return;
    }
    std::vector<std::thread> pool;
    const size_t piece = ((bytes / t) + 4095) & ~(size_t)4095;
    for (int i = 1; i < t; ++i) {
        const size_t off = (size_t)i * piece;
        if (off >= bytes) break;
        const size_t len = std::min(piece, bytes - off);
        pool.emplace_back([=]() { std::memcpy((char *)dst + off, (const char *)src + off, len); });
    }
    std::memcpy(dst, src, std::min(piece, bytes));
    for (std::thread &th : pool) th.join();
}

// Grows the staging ring to `rays_per_slot` rays per slot; the pinned host halves are only allocated when a
// pageable batch needs them.
int ensure_stage(mr_ctx *c, size_t rays_per_slot, bool need_pinned)
{
    const bool have_pinned = c->pinned[0] != nullptr;
    if (c->stage_cap_rays >= rays_per_slot && (have_pinned || !need_pinned)) return MR_OK;
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    MR_CUDA(c, cudaStreamSynchronize(c->copy_stream));
    const size_t cap = std::max(c->stage_cap_rays, rays_per_slot);
    const bool want_pinned = need_pinned || have_pinned;
    free_stage(c);
    const size_t bytes = cap * c->ray_bytes();
    for (int s = 0; s < kStageSlots; ++s) {
        if (want_pinned && cudaMallocHost(&c->pinned[s], bytes) != cudaSuccess) {
            cudaGetLastError();
            free_stage(c);
            return c->fail(MR_ERR_OOM, "pinned host allocation failed (staging ring)");
        }
        c->d_stage[s] = c->dev_alloc(bytes);
        if (!c->d_stage[s]) {
            free_stage(c);
            return c->fail(MR_ERR_OOM, "device allocation failed (staging ring)");
        }
    }
    c->stage_cap_rays = cap;
    return MR_OK;
}

}  // namespace

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

int mr_create_ex(mr_ctx **out, int device, int precision, const mr_allocator *alloc)
{
    if (!out) {
        g_create_error = "out is NULL";
        return MR_ERR_INVALID_ARG;
    }
    *out = nullptr;
    if (precision != MR_PRECISION_MIXED && precision != MR_PRECISION_DOUBLE) {
        g_create_error = "unknown precision mode";
        return MR_ERR_INVALID_ARG;
    }
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess) {
        cudaGetLastError();
        g_create_error = std::string("no usable CUDA device: ") + cudaGetErrorString(e);
        return MR_ERR_CUDA;
    }
    if (device < 0 || device >= count) {
        g_create_error = "device index out of range";
        return MR_ERR_INVALID_ARG;
    }
    if (alloc && (!alloc->alloc || !alloc->free)) {
        g_create_error = "allocator needs both alloc and free";
        return MR_ERR_INVALID_ARG;
    }
    mr_ctx *c = new mr_ctx();
    c->device = device;
    c->precision = precision;
    {
        int l2 = 0;
        if (cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, device) != cudaSuccess) cudaGetLastError();
        c->l2_bytes = (size_t)std::max(l2, 0);
    }
    if (alloc) c->alloc = *alloc;
    DeviceGuard guard(device);
    bool ok = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaStreamCreateWithFlags(&c->stream2, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&c->ev_lane, cudaEventDisableTiming) == cudaSuccess;
    for (int s = 0; s < kStageSlots && ok; ++s) {
        ok = ok && cudaEventCreateWithFlags(&c->ev_copied[s], cudaEventDisableTiming) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&c->ev_done[s], cudaEventDisableTiming) == cudaSuccess;
    }
    ok = ok && cudaEventCreate(&c->ev_t0) == cudaSuccess && cudaEventCreate(&c->ev_t1) == cudaSuccess;
    if (ok) {
        c->d_counters = (unsigned long long *)c->dev_alloc(12 * sizeof(unsigned long long));   // [4..6]: next-event counters; the rest is spare
        ok = c->d_counters && cudaMemset(c->d_counters, 0, 12 * sizeof(unsigned long long)) == cudaSuccess;
    }
    if (!ok) {
        g_create_error = std::string("context set-up failed: ") + cudaGetErrorString(cudaGetLastError());
        mr_destroy(c);
        return MR_ERR_CUDA;
    }
    *out = c;
    return MR_OK;
}

int mr_create(mr_ctx **out, int device, int precision) { return mr_create_ex(out, device, precision, nullptr); }

int mr_destroy(mr_ctx *c)
{
    if (!c) return MR_OK;
    DeviceGuard guard(c->device);
    cudaStreamSynchronize(c->stream);
    if (c->copy_stream) cudaStreamSynchronize(c->copy_stream);
    if (c->stream2) cudaStreamSynchronize(c->stream2);     // before anything its kernels may still read is freed
    if (c->read_stream) {
        cudaStreamSynchronize(c->read_stream);
        cudaStreamDestroy(c->read_stream);
        if (c->ev_snap) cudaEventDestroy(c->ev_snap);
        if (c->ev_read) cudaEventDestroy(c->ev_read);
    }
    c->dev_free(c->d_snap);
    if (c->ring) {
        for (RingSlot *s : c->ring->slots) {
            if (s->ev_copied) { cudaEventSynchronize(s->ev_copied); cudaEventDestroy(s->ev_copied); }
            if (s->ev_done) { cudaEventSynchronize(s->ev_done); cudaEventDestroy(s->ev_done); }
            if (s->pinned) cudaFreeHost(s->pinned);
            delete s;
        }
        if (c->ring->ev_cast) cudaEventDestroy(c->ring->ev_cast);
        c->dev_free(c->ring->d_all);
        delete c->ring;
        c->ring = nullptr;
    }
    free_stage(c);
    for (int b = 0; b < 2; ++b) {
        c->dev_free(c->d_whole[b]);
        if (c->ev_whole_done[b]) cudaEventDestroy(c->ev_whole_done[b]);
    }
    if (c->ev_whole_copied) cudaEventDestroy(c->ev_whole_copied);
    free_tables(c);
    for (int q = 0; q < MR_MAX_NUCLIDES; ++q) {
        unref_grid(c, c->nuc_grid_of[q]);
        c->dev_free(c->nuc_S[q]);
    }
    c->dev_free(c->d_mix_off);
    c->dev_free(c->d_mix_nuc);
    c->dev_free(c->d_mix_w);
    free_materials(c);
    c->dev_free(c->d_edges);
    c->dev_free(c->d_tally);
    c->dev_free(c->d_counters);
    free_defer(c);
    if (c->h_defer_ctl) cudaFreeHost(c->h_defer_ctl);
    if (c->ev_defer) cudaEventDestroy(c->ev_defer);
    c->dev_free(c->d_prev);
    c->dev_free(c->d_s2);
    c->dev_free(c->d_det);
    c->dev_free(c->d_det_sum);
    for (int l = 0; l < 2; ++l) {
        c->dev_free(c->d_keys_l[l]);
        c->dev_free(c->d_perm_l[l]);
        c->dev_free(c->d_hist_l[l]);
        c->dev_free(c->d_blk_hist_l[l]);
    }
    if (c->stream2) { cudaStreamSynchronize(c->stream2); cudaStreamDestroy(c->stream2); }
    if (c->ev_lane) cudaEventDestroy(c->ev_lane);
    for (int s = 0; s < kStageSlots; ++s) {
        if (c->ev_copied[s]) cudaEventDestroy(c->ev_copied[s]);
        if (c->ev_done[s]) cudaEventDestroy(c->ev_done[s]);
    }
    for (cudaEvent_t e : c->kev) cudaEventDestroy(e);
    if (c->ev_t0) cudaEventDestroy(c->ev_t0);
    if (c->ev_t1) cudaEventDestroy(c->ev_t1);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    cudaGetLastError();
    delete c;
    return MR_OK;
}

int mr_set_stream(mr_ctx *c, void *cuda_stream)
{
    MR_ENTER(c);
    if (c->ring) return c->fail(MR_ERR_STATE, "set_stream: close the producer ring first (its pushes queue work on the stream)");
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    MR_CUDA(c, cudaStreamSynchronize(c->copy_stream));
    if (c->stream2) MR_CUDA(c, cudaStreamSynchronize(c->stream2));
    if (c->read_stream) MR_CUDA(c, cudaStreamSynchronize(c->read_stream));
    c->read_pending = false;
    c->stream = (cudaStream_t)cuda_stream;
    return MR_OK;
}

const char *mr_last_error(mr_ctx *c) { return c ? c->err.c_str() : g_create_error.c_str(); }

}  // extern "C"

namespace {

int load_mesh_common(mr_ctx *c, bool rz, int nx, int ny, int nz, const double *xe, const double *ye, const double *ze)
{
    if (nx < 1 || ny < 1 || nz < 1 || !xe || !ye || !ze) return c->fail(MR_ERR_INVALID_ARG, "mesh: bad size or NULL edge array");
    const long long ncell = (long long)nx * ny * nz;
    if ((long long)nx * ny > 0x7fffffffLL || ncell >= 0x7fffffffLL) return c->fail(MR_ERR_UNSUPPORTED, "mesh: nx*ny*nz must be < 2^31");
    if (nx > 32767 || ny > 32767 || nz > 32767) return c->fail(MR_ERR_UNSUPPORTED, "mesh: at most 32767 cells per axis");
    if (!finite_increasing(xe, nx + 1) || !finite_increasing(ye, ny + 1) || !finite_increasing(ze, nz + 1))
        return c->fail(MR_ERR_INVALID_ARG, "mesh: plane positions must be finite and strictly increasing");
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    if (c->stream2) MR_CUDA(c, cudaStreamSynchronize(c->stream2));
    free_materials(c);
    // the deferred tally's chunk table is laid out for the regions of ONE mesh (nbin rows), and its pool estimate is that
    // mesh's segments per ray: a new mesh starts from nothing
    free_defer(c);
    c->defer_entries_per_ray = 0.0;
    c->defer_direct_seen = 0;
    c->dev_free(c->d_edges);
    c->dev_free(c->d_tally);
    c->dev_free(c->d_prev);
    c->dev_free(c->d_s2);
    if (c->read_stream) cudaStreamSynchronize(c->read_stream);
    c->read_pending = false;
    c->dev_free(c->d_snap);
    c->d_snap = nullptr;
    c->d_edges = nullptr;
    c->d_tally = nullptr;
    c->d_prev = c->d_s2 = nullptr;
    c->nbatch = 0;
    c->tally_borrowed = false;
    const int ne = nx + ny + nz + 3;
    std::vector<double> h(ne);
    std::memcpy(h.data(), xe, sizeof(double) * (nx + 1));
    std::memcpy(h.data() + nx + 1, ye, sizeof(double) * (ny + 1));
    std::memcpy(h.data() + nx + ny + 2, ze, sizeof(double) * (nz + 1));
    c->d_edges = (double *)c->dev_alloc(sizeof(double) * ne);
    c->d_tally = (double *)c->dev_alloc(sizeof(double) * ncell);
    if (!c->d_edges || !c->d_tally) {
        c->dev_free(c->d_edges);
        c->dev_free(c->d_tally);
        c->d_edges = nullptr;
        c->d_tally = nullptr;
        return c->fail(MR_ERR_OOM, "device allocation failed (mesh / tally)");
    }
    c->nx = nx; c->ny = ny; c->nz = nz; c->nedges = ne; c->ncell = ncell;
    c->mesh_rz = rz;
    c->mesh_sphere = false;
    {   // arithmetic mesh?  (uniform spacing reproduced exactly by one fma per plane, checked plane by plane)
        const double *ax[3] = {xe, ye, ze};
        const int na[3] = {nx, ny, nz};
        c->mesh_arith = true;
        for (int a = 0; a < 3; ++a) {
            c->mesh_e0[a] = ax[a][0];
            c->mesh_h[a] = ax[a][1] - ax[a][0];
            for (int p = 0; p <= na[a] && c->mesh_arith; ++p)
                c->mesh_arith = (std::fma((double)p, c->mesh_h[a], c->mesh_e0[a]) == ax[a][p]);
        }
        if (rz) c->mesh_arith = false;   // the R-Z walker reads its radii and planes from the table
    }
    MR_CUDA(c, cudaMemcpyAsync(c->d_edges, h.data(), sizeof(double) * ne, cudaMemcpyHostToDevice, c->stream));
    MR_CUDA(c, cudaMemsetAsync(c->d_tally, 0, sizeof(double) * ncell, c->stream));
    MR_CUDA(c, cudaMemsetAsync(c->d_counters, 0, 4 * sizeof(unsigned long long), c->stream));
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    return MR_OK;
}

}  // namespace

extern "C" {

int mr_load_mesh(mr_ctx *c, int nx, int ny, int nz, const double *xe, const double *ye, const double *ze)
{
    MR_ENTER(c);
    MR_NO_RING(c, "mr_load_mesh");
    return load_mesh_common(c, false, nx, ny, nz, xe, ye, ze);
}

int mr_load_mesh_rz(mr_ctx *c, int nr, int nz, const double *re, const double *ze)
{
    MR_ENTER(c);
    MR_NO_RING(c, "mr_load_mesh_rz");
    if (nr < 1 || !re) return c->fail(MR_ERR_INVALID_ARG, "rz mesh: bad size or NULL radius array");
    if (re[0] != 0.0) return c->fail(MR_ERR_INVALID_ARG, "rz mesh: the first radius must be 0");
    const double ye[2] = {0.0, 1.0};
    return load_mesh_common(c, true, nr, 1, nz, re, ye, ze);
}

int mr_load_mesh_sphere(mr_ctx *c, int nr, const double *re)
{
    MR_ENTER(c);
    MR_NO_RING(c, "mr_load_mesh_sphere");
    if (nr < 1 || !re) return c->fail(MR_ERR_INVALID_ARG, "spherical mesh: bad size or NULL radius array");
    if (re[0] != 0.0) return c->fail(MR_ERR_INVALID_ARG, "spherical mesh: the first radius must be 0");
    const double one[2] = {0.0, 1.0};
    if (int rc = load_mesh_common(c, true, nr, 1, 1, re, one, one)) return rc;
    c->mesh_sphere = true;
    return MR_OK;
}

int mr_load_materials(mr_ctx *c, int M, const double *density, int K, const int32_t *cell_mat, const double *cell_frac)
{
    MR_ENTER(c);
    MR_NO_RING(c, "mr_load_materials");
    if (!c->d_tally) return c->fail(MR_ERR_STATE, "load the mesh before the materials");
    if (M < 1 || K < 1 || !density || !cell_mat || !cell_frac) return c->fail(MR_ERR_INVALID_ARG, "materials: bad size or NULL array");
    if (M > MR_MAX_MATERIALS) return c->fail(MR_ERR_UNSUPPORTED, "materials: M > MR_MAX_MATERIALS");
    if (K > MR_MAX_SLOTS) return c->fail(MR_ERR_UNSUPPORTED, "materials: K > MR_MAX_SLOTS");
    for (int m = 0; m < M; ++m)
        if (!std::isfinite(density[m]) || density[m] < 0.0) return c->fail(MR_ERR_INVALID_ARG, "materials: densities must be finite and >= 0");
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    if (M != c->M) free_tables(c);
    free_materials(c);

    const bool dbl = c->precision == MR_PRECISION_DOUBLE;
    int layout = LAYOUT_GENERIC;
    if (dbl && K <= 3) layout = LAYOUT_DK3;
    if (!dbl) {
        if (K <= 4) layout = K;  // LAYOUT_K1..K4
        if (K == 8 && M == 8) {  // dense: every cell lists materials 0..7 in order (ids implicit)
            bool dense = true;
            for (long long i = 0; i < c->ncell * 8 && dense; ++i) dense = cell_mat[i] == (int32_t)(i & 7);
            if (dense) layout = LAYOUT_D8;
        }
    }
    size_t rec_bytes = 0, id_bytes = 0;
    switch (layout) {
    case LAYOUT_K1: rec_bytes = 8; break;
    case LAYOUT_K2: case LAYOUT_K3: rec_bytes = 16; break;
    case LAYOUT_K4: case LAYOUT_D8: case LAYOUT_DK3: rec_bytes = 32; break;
    default: rec_bytes = (size_t)K * (dbl ? 8 : 4); id_bytes = (size_t)K;
    }
    const long long chunk = std::min<long long>(c->ncell, 1LL << 22);
    void *recs = c->dev_alloc(rec_bytes * (c->ncell + 4));   // + 4: 16-byte records are read as aligned pairs, 8-byte ones in fours
    uint8_t *ids = id_bytes ? (uint8_t *)c->dev_alloc(id_bytes * c->ncell) : nullptr;
    int32_t *s_mat = (int32_t *)c->dev_alloc(sizeof(int32_t) * chunk * K);
    double *s_frac = (double *)c->dev_alloc(sizeof(double) * chunk * K);
    double *s_den = (double *)c->dev_alloc(sizeof(double) * M);
    int *s_flags = (int *)c->dev_alloc(sizeof(int));
    auto cleanup = [&](bool all) {
        c->dev_free(s_mat); c->dev_free(s_frac); c->dev_free(s_den); c->dev_free(s_flags);
        if (all) { c->dev_free(recs); c->dev_free(ids); }
    };
    if (!recs || (id_bytes && !ids) || !s_mat || !s_frac || !s_den || !s_flags) {
        cleanup(true);
        return c->fail(MR_ERR_OOM, "device allocation failed (cell records)");
    }
    cudaError_t e = cudaMemcpyAsync(s_den, density, sizeof(double) * M, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(s_flags, 0, sizeof(int), c->stream);
    for (long long first = 0; first < c->ncell && e == cudaSuccess; first += chunk) {
        const long long count = std::min(chunk, c->ncell - first);
        e = cudaMemcpyAsync(s_mat, cell_mat + first * K, sizeof(int32_t) * count * K, cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(s_frac, cell_frac + first * K, sizeof(double) * count * K, cudaMemcpyHostToDevice, c->stream);
        if (e != cudaSuccess) break;
        PackParams P{s_mat, s_frac, s_den, first, count, K, M, layout, dbl ? 1 : 0, recs, ids, s_flags};
        pack_cells_kernel<<<(unsigned)((count + 255) / 256), 256, 0, c->stream>>>(P);
        c->launches += 1;
        e = cudaGetLastError();
        // the pageable source is consumed when the copy call returns; the scratch is reused in stream order
    }
    int flags = 0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&flags, s_flags, sizeof(int), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) {
        cleanup(true);
        return c->fail_cuda(e, "mr_load_materials");
    }
    if (flags) {
        cleanup(true);
        return c->fail(MR_ERR_INVALID_ARG, (flags & 1) ? "materials: cell_mat entry outside [-1, M)" : "materials: cell_frac must be finite and >= 0");
    }
    cleanup(false);
    c->d_recs = recs;
    c->d_ids = ids;
    c->layout = layout;
    c->rec_bytes_per_cell = rec_bytes + id_bytes;
    c->fused = layout == LAYOUT_K4 && !c->mesh_rz &&
               (c->fused_opt == 1 || (c->fused_opt == 2 && (size_t)c->ncell * 40 > 2 * c->l2_bytes));
    c->fused_dirty = false;
    c->K = K;
    if (int rc = build_tiled_index(c, M, density, K, cell_mat, cell_frac)) return rc;
    if (c->ndict == 0) {
        if (int rc = build_coarse_records(c, density, K, cell_mat, cell_frac)) return rc;
    }
    if (c->cshift > 0) c->fused = false;     // the records are no longer per cell: nowhere to keep a per-cell accumulator
    if (M != c->M || (int)c->xs_n.size() != M) {
        c->M = M;
        c->mix.assign(M, {});
        c->grid_of.assign(M, nullptr);
        c->d_S.assign(M, nullptr);
        c->xs_n.assign(M, 0);
        c->xs_dirty = true;
    }
    return MR_OK;
}

}  // extern "C"

namespace {

// Validates and uploads one (energy, sigma) table into the given slot (a material's or a nuclide's).
int load_table(mr_ctx *c, mr_ctx::Grid **grid_slot, void **S_slot, int *n_slot, int64_t n, const double *energy,
               const double *sigma_t)
{
    const bool dbl = c->precision == MR_PRECISION_DOUBLE;
    std::vector<float> ef, sf;
    if (!dbl) { ef.resize(n); sf.resize(n); }
    for (int64_t i = 0; i < n; ++i) {
        if (!std::isfinite(energy[i]) || !(energy[i] > 0.0) || !std::isfinite(sigma_t[i]) || sigma_t[i] < 0.0)
            return c->fail(MR_ERR_INVALID_ARG, "xs: energies must be finite and > 0, cross sections finite and >= 0");
        if (!dbl) {
            ef[i] = (float)energy[i];
            sf[i] = (float)sigma_t[i];
            if (!std::isfinite(ef[i]) || !std::isfinite(sf[i]) || !(ef[i] > 0.f))
                return c->fail(MR_ERR_INVALID_ARG, "xs: value not representable in fp32");
            if (i && !(ef[i] > ef[i - 1])) return c->fail(MR_ERR_INVALID_ARG, "xs: energy grid not strictly increasing (after fp32 rounding)");
        } else if (i && !(energy[i] > energy[i - 1]))
            return c->fail(MR_ERR_INVALID_ARG, "xs: energy grid not strictly increasing");
    }
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    const size_t bytes = (size_t)n * c->real_bytes();
    const void *hE = dbl ? (const void *)energy : (const void *)ef.data();
    const void *hS = dbl ? (const void *)sigma_t : (const void *)sf.data();

    // the energy grid: reuse a resident one if it is bitwise identical, else upload it with its bucket index
    mr_ctx::Grid *g = nullptr;
    for (mr_ctx::Grid *q : c->grids)
        if (q->n == (int)n && q->host.size() == bytes && std::memcmp(q->host.data(), hE, bytes) == 0) { g = q; break; }
    bool new_grid = false;
    std::vector<uint32_t> first;
    if (!g) {
        new_grid = true;
        g = new mr_ctx::Grid();
        g->n = (int)n;
        g->host.assign((const unsigned char *)hE, (const unsigned char *)hE + bytes);
        // bucket(E) = (bits((float)E) >> sh) - b0: positive floats order like their bit patterns and double -> float
        // rounding is monotone, so bucket() is non-decreasing in E in both precision modes
        auto fbits = [&](int64_t i) {
            const float f = dbl ? (float)energy[i] : ef[i];
            uint32_t u;
            std::memcpy(&u, &f, 4);
            return u;
        };
        const uint32_t lo_bits = fbits(0), hi_bits = fbits(n - 1);
        const uint64_t want = std::min<uint64_t>(std::max<uint64_t>(2 * (uint64_t)n, 1024), 1u << 20);
        int sh = 0;
        while ((uint64_t)(hi_bits >> sh) - (lo_bits >> sh) + 1 > want) ++sh;
        g->sh = sh;
        g->b0 = lo_bits >> sh;
        const uint32_t nb = (hi_bits >> sh) - g->b0 + 1;
        first.assign((size_t)nb + 1, 0);
        for (int64_t i = 0; i < n; ++i) first[(fbits(i) >> sh) - g->b0 + 1] += 1;   // counts, shifted by one
        for (uint32_t b2 = 0; b2 < nb; ++b2) first[b2 + 1] += first[b2];            // first[b] = #points with bucket < b
        g->d_E = c->dev_alloc(bytes);
        g->d_first = (uint32_t *)c->dev_alloc(first.size() * sizeof(uint32_t));
    }
    void *dS = c->dev_alloc(bytes);
    auto drop_new = [&]() {
        if (new_grid) {
            c->dev_free(g->d_E);
            c->dev_free(g->d_first);
            delete g;
        }
        c->dev_free(dS);
    };
    if (!dS || !g->d_E || !g->d_first) {
        drop_new();
        return c->fail(MR_ERR_OOM, "device allocation failed (cross-section table)");
    }
    cudaError_t e = cudaMemcpyAsync(dS, hS, bytes, cudaMemcpyHostToDevice, c->stream);
    if (new_grid && e == cudaSuccess) e = cudaMemcpyAsync(g->d_E, hE, bytes, cudaMemcpyHostToDevice, c->stream);
    if (new_grid && e == cudaSuccess)
        e = cudaMemcpyAsync(g->d_first, first.data(), first.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) {
        drop_new();
        return c->fail_cuda(e, "mr_load_xs");
    }
    if (new_grid) {
        g->id = c->next_grid_id++;
        c->grids.push_back(g);
    }
    g->refs += 1;
    unref_grid(c, *grid_slot);   // the table this call replaces, if any
    c->dev_free(*S_slot);
    *grid_slot = g;
    *S_slot = dS;
    *n_slot = (int)n;
    c->xs_dirty = true;
    return MR_OK;
}
}  // namespace

extern "C" {

int mr_load_xs(mr_ctx *c, int material, int64_t n, const double *energy, const double *sigma_t)
{
    MR_ENTER(c);
    MR_NO_RING(c, "mr_load_xs");
    if (!c->d_recs) return c->fail(MR_ERR_STATE, "load the materials before the tables");
    if (material < 0 || material >= c->M || n < 1 || n > 0x7fffffff || !energy || !sigma_t)
        return c->fail(MR_ERR_INVALID_ARG, "xs: bad material index, size or NULL array");
    if (int rc = load_table(c, &c->grid_of[material], &c->d_S[material], &c->xs_n[material], n, energy, sigma_t)) return rc;
    c->mix[material].clear();       // a table of its own replaces a nuclide mixture
    return MR_OK;
}

int mr_load_nuclide_xs(mr_ctx *c, int nuclide, int64_t n, const double *energy, const double *sigma)
{
    MR_ENTER(c);
    MR_NO_RING(c, "mr_load_nuclide_xs");
    if (nuclide < 0 || nuclide >= MR_MAX_NUCLIDES || n < 1 || n > 0x7fffffff || !energy || !sigma)
        return c->fail(MR_ERR_INVALID_ARG, "nuclide xs: bad nuclide index, size or NULL array");
    return load_table(c, &c->nuc_grid_of[nuclide], &c->nuc_S[nuclide], &c->nuc_n[nuclide], n, energy, sigma);
}

int mr_define_material(mr_ctx *c, int material, int nnuc, const int32_t *nuclides, const double *weights)
{
    MR_ENTER(c);
    MR_NO_RING(c, "mr_define_material");
    if (!c->d_recs) return c->fail(MR_ERR_STATE, "load the materials before defining their composition");
    if (material < 0 || material >= c->M || nnuc < 1 || nnuc > MR_MAX_MIX || !nuclides || !weights)
        return c->fail(MR_ERR_INVALID_ARG, "define_material: bad material index, nuclide count or NULL array");
    std::vector<std::pair<int, double>> mix;
    for (int j = 0; j < nnuc; ++j) {
        if (nuclides[j] < 0 || nuclides[j] >= MR_MAX_NUCLIDES) return c->fail(MR_ERR_INVALID_ARG, "define_material: nuclide index out of range");
        if (!std::isfinite(weights[j]) || weights[j] < 0.0 || (c->precision == MR_PRECISION_MIXED && !std::isfinite((float)weights[j])))
            return c->fail(MR_ERR_INVALID_ARG, "define_material: weights must be finite and >= 0");
        mix.emplace_back(nuclides[j], weights[j]);
    }
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    unref_grid(c, c->grid_of[material]);    // the mixture replaces a table of its own
    c->dev_free(c->d_S[material]);
    c->grid_of[material] = nullptr;
    c->d_S[material] = nullptr;
    c->xs_n[material] = 0;
    c->mix[material] = mix;
    c->xs_dirty = true;
    return MR_OK;
}

}  // extern "C"

namespace {

// Runs `work(count, device rays)` over a batch: a device batch in one piece, a host batch in staged chunks.
// one_lane: the work keeps per-context device state that two chunks in flight would share (the deferred tally's control
// words, chunk table and pool): its chunks stay on the context's stream, one after the other.
template <typename Work>
int run_batch(mr_ctx *c, int64_t n, const void *rays, int where, Work work, bool one_lane = false)
{
    c->kev_used = 0;
    if (where == MR_WHERE_DEVICE) {
        if ((uintptr_t)rays & 15) return c->fail(MR_ERR_INVALID_ARG, "cast: device ray buffer must be 16-byte aligned");
        MR_CUDA(c, cudaEventRecord(c->ev_t0, c->stream));
        if (int rc = work((long long)n, rays)) return rc;
        MR_CUDA(c, cudaEventRecord(c->ev_t1, c->stream));
        c->have_timing = true;
        return MR_OK;
    }
    // Host batch, in chunks of MR_OPT_STAGE_RAYS rays through a 2-slot device ring: the H2D copy of chunk i+1
    // (copy stream) overlaps the kernels of chunk i (context stream) -- the CPU/GPU overlap of Fig. 4
    // inside one call.  A pinned (page-locked) caller buffer is the DMA source itself; a
    // pageable one is first copied, by a few host threads, into a pinned ring slot.
    const size_t rb = c->ray_bytes();
    const size_t per = (size_t)std::max<long long>(1024, std::min<long long>(c->stage_rays, n));
    bool pinned_src = false;
    {
        cudaPointerAttributes at{};
        if (cudaPointerGetAttributes(&at, rays) == cudaSuccess) pinned_src = (at.type == cudaMemoryTypeHost);
        else cudaGetLastError();
        if (pinned_src) {   // the whole batch must lie inside the registered range
            cudaPointerAttributes at2{};
            const char *last = (const char *)rays + (size_t)n * rb - 1;
            if (cudaPointerGetAttributes(&at2, last) != cudaSuccess || at2.type != cudaMemoryTypeHost) {
                cudaGetLastError();
                pinned_src = false;
            }
        }
    }
    // Back-to-back host batches: when the context's stream is still busy with earlier work (a caller that casts batch after
    // batch without waiting), the chunked pipeline below buys nothing -- its point is to start the first kernel early on an
    // IDLE GPU -- and costs 20 % in kernel time (chunks of 2^18..2^21 rays are cast less efficiently than the batch in one
    // launch).  Then the whole batch is DMA'd into one of two device buffers while the earlier work runs, and cast in one
    // launch behind it: in steady state the copy of batch i+1 hides behind the cast of batch i.
    constexpr size_t kWholeMaxBytes = (size_t)2 << 30;
    bool stream_busy = false;
    if (c->whole_opt == 2) {
        stream_busy = cudaStreamQuery(c->stream) == cudaErrorNotReady;
        cudaGetLastError();
    }
    if (pinned_src && (c->whole_opt == 1 || stream_busy) && (size_t)n * rb <= kWholeMaxBytes && (size_t)n > per) {
        const size_t bytes = (size_t)n * rb;
        if (!c->ev_whole_copied) {
            MR_CUDA(c, cudaEventCreateWithFlags(&c->ev_whole_copied, cudaEventDisableTiming));
            for (int b = 0; b < 2; ++b) MR_CUDA(c, cudaEventCreateWithFlags(&c->ev_whole_done[b], cudaEventDisableTiming));
        }
        if (bytes > c->whole_cap_bytes) {
            MR_CUDA(c, cudaStreamSynchronize(c->stream));
            MR_CUDA(c, cudaStreamSynchronize(c->copy_stream));
            for (int b = 0; b < 2; ++b) {
                c->dev_free(c->d_whole[b]);
                c->d_whole[b] = c->dev_alloc(bytes);
            }
            c->whole_cap_bytes = (c->d_whole[0] && c->d_whole[1]) ? bytes : 0;
            if (!c->whole_cap_bytes) {
                for (int b = 0; b < 2; ++b) { c->dev_free(c->d_whole[b]); c->d_whole[b] = nullptr; }
                return c->fail(MR_ERR_OOM, "device allocation failed (whole-batch staging)");
            }
        }
        const int b = c->whole_next;
        c->whole_next ^= 1;
        MR_CUDA(c, cudaEventRecord(c->ev_t0, c->stream));
        MR_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->ev_whole_done[b], 0));   // the cast that last read this buffer is done
        MR_CUDA(c, cudaMemcpyAsync(c->d_whole[b], rays, bytes, cudaMemcpyHostToDevice, c->copy_stream));
        MR_CUDA(c, cudaEventRecord(c->ev_whole_copied, c->copy_stream));
        MR_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_whole_copied, 0));
        if (int rc = work((long long)n, (const void *)c->d_whole[b])) return rc;
        MR_CUDA(c, cudaEventRecord(c->ev_whole_done[b], c->stream));
        MR_CUDA(c, cudaEventRecord(c->ev_t1, c->stream));
        c->have_timing = true;
        MR_CUDA(c, cudaEventSynchronize(c->ev_whole_copied));      // the caller's buffer is consumed when the call returns
        return MR_OK;
    }
    // Chunk sizes grow: per/4, per/2, per, 2 per, 2 per, ...  The first copy is short, so the first kernel starts
    // early, and the later chunks are large, where the ordering pre-pass keeps the cast kernel's working set in L2
    // (a 2^18-ray chunk costs 2.8x more per ray than a 10^7-ray batch on the PWR-like config).
    const size_t big = (size_t)n > 2 * per ? 2 * per : per;
    if (int rc = ensure_stage(c, big, !pinned_src)) return rc;
    MR_CUDA(c, cudaEventRecord(c->ev_t0, c->stream));
    int64_t chunk = (int64_t)std::max<size_t>(1024, (size_t)n > 2 * per ? per / 4 : per);
    int last_slot = -1;
    // Consecutive chunks alternate between the two compute lanes: every cast kernel ramps up and down for about
    // 0.2 ms (a CTA lives as long as its longest ray), and with one stream those ramps add up chunk after chunk.
    // (Not on R-Z meshes: their persistent kernel has one work counter.  Not with the deferred tally: see one_lane.)
    const bool two_lanes = !c->mesh_rz && !one_lane && n > chunk;
    // on EVERY exit path (errors included) lane 1 is joined back into the context's stream: work the caller queues there
    // afterwards, and the frees of mr_destroy, come after everything this call launched
    struct LaneReset {
        mr_ctx *c;
        bool forked = false;
        void join()
        {
            c->lane = 0;
            if (forked) {
                forked = false;
                if (cudaEventRecord(c->ev_lane, c->stream2) == cudaSuccess) cudaStreamWaitEvent(c->stream, c->ev_lane, 0);
                else cudaGetLastError();
            }
        }
        ~LaneReset() { join(); }
    } lane_reset{c};
    if (two_lanes) {
        MR_CUDA(c, cudaEventRecord(c->ev_lane, c->stream));
        MR_CUDA(c, cudaStreamWaitEvent(c->stream2, c->ev_lane, 0));
        lane_reset.forked = true;
    }
    int k = 0;
    for (int64_t first = 0, count = 0; first < n; first += count, chunk = std::min<int64_t>(2 * chunk, (int64_t)big), ++k) {
        count = std::min<int64_t>(chunk, n - first);
        c->lane = two_lanes ? (k & 1) : 0;
        const int s = c->next_slot;
        c->next_slot = (s + 1) % kStageSlots;
        const char *src = (const char *)rays + (size_t)first * rb;
        if (!pinned_src) {
            MR_CUDA(c, cudaEventSynchronize(c->ev_copied[s]));       // pinned slot free again
            host_copy(c->pinned[s], src, (size_t)count * rb, c->copy_threads);
            src = (const char *)c->pinned[s];
        }
        MR_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->ev_done[s], 0));  // device slot free again
        MR_CUDA(c, cudaMemcpyAsync(c->d_stage[s], src, (size_t)count * rb, cudaMemcpyHostToDevice, c->copy_stream));
        MR_CUDA(c, cudaEventRecord(c->ev_copied[s], c->copy_stream));
        MR_CUDA(c, cudaStreamWaitEvent(c->work_stream(), c->ev_copied[s], 0));
        if (int rc = work((long long)count, (const void *)c->d_stage[s])) return rc;
        MR_CUDA(c, cudaEventRecord(c->ev_done[s], c->work_stream()));
        last_slot = s;
    }
    lane_reset.join();   // the context's stream continues after both lanes
    MR_CUDA(c, cudaEventRecord(c->ev_t1, c->stream));
    c->have_timing = true;
    // the caller's buffer is consumed when the call returns: wait for the last DMA out of it
    if (pinned_src && last_slot >= 0) MR_CUDA(c, cudaEventSynchronize(c->ev_copied[last_slot]));
    return MR_OK;
}

}  // namespace

extern "C" {

int mr_cast_rays(mr_ctx *c, int64_t n, const void *rays, int where)
{
    MR_ENTER(c);
    if (n < 0 || (n > 0 && !rays) || (where != MR_WHERE_HOST && where != MR_WHERE_DEVICE))
        return c->fail(MR_ERR_INVALID_ARG, "cast: bad count, NULL buffer or unknown location");
    if (int rc = ready_to_cast(c)) return rc;
    if (n == 0) return MR_OK;
    if (int rc = upload_xs_desc(c)) return rc;
    return run_batch(c, n, rays, where, [c](long long count, const void *d_rays) { return cast_device(c, count, d_rays); },
                     use_deferred(c, record_path(c)));
}

int mr_read_tally(mr_ctx *c, double *out)
{
    MR_ENTER(c);
    if (!out) return c->fail(MR_ERR_INVALID_ARG, "read_tally: out is NULL");
    if (!c->d_tally) return c->fail(MR_ERR_STATE, "no mesh loaded");
    MR_CUDA(c, flush_accumulators(c));
    MR_CUDA(c, cudaMemcpyAsync(out, c->d_tally, sizeof(double) * c->ncell, cudaMemcpyDeviceToHost, c->stream));
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    if (c->read_stream && c->read_pending) {       // earlier mr_read_tally_async transfers are complete too
        MR_CUDA(c, cudaStreamSynchronize(c->read_stream));
        c->read_pending = false;
    }
    return MR_OK;
}

int mr_clear_tally(mr_ctx *c)
{
    MR_ENTER(c);
    if (!c->d_tally) return c->fail(MR_ERR_STATE, "no mesh loaded");
    MR_CUDA(c, flush_accumulators(c));      // empties the in-record accumulators
    MR_CUDA(c, cudaMemsetAsync(c->d_tally, 0, sizeof(double) * c->ncell, c->stream));
    MR_CUDA(c, cudaMemsetAsync(c->d_counters, 0, 4 * sizeof(unsigned long long), c->stream));
    if (c->d_prev) {   // the batch moments restart with the tally
        MR_CUDA(c, cudaMemsetAsync(c->d_prev, 0, sizeof(double) * c->ncell, c->stream));
        MR_CUDA(c, cudaMemsetAsync(c->d_s2, 0, sizeof(double) * c->ncell, c->stream));
    }
    c->nbatch = 0;
    return MR_OK;
}

int mr_sync(mr_ctx *c)
{
    MR_ENTER(c);
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    if (c->read_stream && c->read_pending) {
        MR_CUDA(c, cudaStreamSynchronize(c->read_stream));
        c->read_pending = false;
    }
    return MR_OK;
}

int mr_read_tally_async(mr_ctx *c, double *out)
{
    MR_ENTER(c);
    if (!out) return c->fail(MR_ERR_INVALID_ARG, "read_tally_async: out is NULL");
    if (!c->d_tally) return c->fail(MR_ERR_STATE, "no mesh loaded");
    if (!c->read_stream) {
        MR_CUDA(c, cudaStreamCreateWithFlags(&c->read_stream, cudaStreamNonBlocking));
        MR_CUDA(c, cudaEventCreateWithFlags(&c->ev_snap, cudaEventDisableTiming));
        MR_CUDA(c, cudaEventCreateWithFlags(&c->ev_read, cudaEventDisableTiming));
    }
    if (!c->d_snap) {
        c->d_snap = (double *)c->dev_alloc(sizeof(double) * c->ncell);
        if (!c->d_snap) return c->fail(MR_ERR_OOM, "device allocation failed (tally snapshot)");
    }
    MR_CUDA(c, flush_accumulators(c));
    // the snapshot is taken in stream order (after everything queued so far, before anything queued later); the previous
    // read, if any, must have left the snapshot buffer
    if (c->read_pending) MR_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_read, 0));
    MR_CUDA(c, cudaMemcpyAsync(c->d_snap, c->d_tally, sizeof(double) * c->ncell, cudaMemcpyDeviceToDevice, c->stream));
    MR_CUDA(c, cudaEventRecord(c->ev_snap, c->stream));
    MR_CUDA(c, cudaStreamWaitEvent(c->read_stream, c->ev_snap, 0));
    MR_CUDA(c, cudaMemcpyAsync(out, c->d_snap, sizeof(double) * c->ncell, cudaMemcpyDeviceToHost, c->read_stream));
    MR_CUDA(c, cudaEventRecord(c->ev_read, c->read_stream));
    c->read_pending = true;
    return MR_OK;
}

int mr_get_stats(mr_ctx *c, mr_stats *out)
{
    MR_ENTER(c);
    if (!out) return c->fail(MR_ERR_INVALID_ARG, "get_stats: out is NULL");
    unsigned long long h[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    MR_CUDA(c, cudaMemcpyAsync(h, c->d_counters, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    std::memset(out, 0, sizeof(*out));
    out->rays_accepted = (int64_t)h[0];
    out->rays_rejected = (int64_t)h[1];
    out->segments = (int64_t)h[2];
    out->ne_pairs_accepted = (int64_t)h[4];
    out->ne_pairs_rejected = (int64_t)h[5];
    out->ne_segments = (int64_t)h[6];
    out->kernel_launches = c->launches;
    if (c->have_timing) {
        float ms = 0.f;
        MR_CUDA(c, cudaEventElapsedTime(&ms, c->ev_t0, c->ev_t1));
        out->last_cast_ms = ms;
        for (size_t i = 0; i + 1 < c->kev_used; i += 2) {
            MR_CUDA(c, cudaEventElapsedTime(&ms, c->kev[i], c->kev[i + 1]));
            out->last_kernel_ms += ms;
        }
    }
    return MR_OK;
}

int mr_tally_device_ptr(mr_ctx *c, double **out)
{
    MR_ENTER(c);
    if (!out) return c->fail(MR_ERR_INVALID_ARG, "tally_device_ptr: out is NULL");
    if (!c->d_tally) return c->fail(MR_ERR_STATE, "no mesh loaded");
    MR_CUDA(c, flush_accumulators(c));
    c->tally_borrowed = true;
    *out = c->d_tally;
    return MR_OK;
}

int mr_trace_rays(mr_ctx *c, int64_t n, const void *rays, int where, uint32_t *nseg, uint64_t *hash, int32_t *cells,
                  double *lens, int64_t cap)
{
    MR_ENTER(c);
    if (n < 0 || (n > 0 && !rays) || cap < 0 || (where != MR_WHERE_HOST && where != MR_WHERE_DEVICE))
        return c->fail(MR_ERR_INVALID_ARG, "trace: bad count, NULL buffer or unknown location");
    if (!c->d_tally) return c->fail(MR_ERR_STATE, "no mesh loaded");
    if (n == 0) return MR_OK;
    if (!cells && !lens) cap = 0;
    const size_t rb = c->ray_bytes();
    void *d_rays = nullptr;
    uint32_t *d_nseg = nullptr;
    unsigned long long *d_hash = nullptr;
    int32_t *d_cells = nullptr;
    double *d_lens = nullptr;
    auto cleanup = [&]() {
        if (where == MR_WHERE_HOST) c->dev_free(d_rays);
        c->dev_free(d_nseg); c->dev_free(d_hash); c->dev_free(d_cells); c->dev_free(d_lens);
    };
    bool ok = true;
    if (where == MR_WHERE_HOST) ok = ok && (d_rays = c->dev_alloc((size_t)n * rb));
    if (nseg) ok = ok && (d_nseg = (uint32_t *)c->dev_alloc((size_t)n * 4));
    if (hash) ok = ok && (d_hash = (unsigned long long *)c->dev_alloc((size_t)n * 8));
    if (cells && cap) ok = ok && (d_cells = (int32_t *)c->dev_alloc((size_t)n * cap * 4));
    if (lens && cap) ok = ok && (d_lens = (double *)c->dev_alloc((size_t)n * cap * 8));
    if (!ok) {
        cleanup();
        return c->fail(MR_ERR_OOM, "device allocation failed (trace buffers)");
    }
    cudaError_t e = cudaSuccess;
    if (where == MR_WHERE_HOST) e = cudaMemcpyAsync(d_rays, rays, (size_t)n * rb, cudaMemcpyHostToDevice, c->stream);
    else {
        if ((uintptr_t)rays & 15) { cleanup(); return c->fail(MR_ERR_INVALID_ARG, "trace: device ray buffer must be 16-byte aligned"); }
        d_rays = const_cast<void *>(rays);
    }
    // cells/lens beyond nseg stay as the caller left them: seed the device copies from the host arrays
    if (e == cudaSuccess && d_cells) e = cudaMemcpyAsync(d_cells, cells, (size_t)n * cap * 4, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess && d_lens) e = cudaMemcpyAsync(d_lens, lens, (size_t)n * cap * 8, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess && c->mesh_rz) {
        RzParams Q{};
        Q.c.mesh = mesh_dev(c);
        Q.c.rays = d_rays;
        Q.c.n = n;
        Q.c.counters = c->d_counters;     // only the work counter [3] is used by a trace launch
        Q.nseg = d_nseg; Q.hash = d_hash; Q.cells = d_cells; Q.lens = d_lens; Q.cap = cap;
        Q.ray_is_double = c->precision == MR_PRECISION_DOUBLE ? 1 : 0;
        Q.spherical = c->mesh_sphere ? 1 : 0;
        if (launch_rz_t<float, CellRecGeneric<float>, true>(c, Q, 256) != MR_OK) { cleanup(); return MR_ERR_CUDA; }
    } else if (e == cudaSuccess) {
        TraceParams P{mesh_dev(c), d_rays, n, d_nseg, d_hash, d_cells, d_lens, cap, c->precision == MR_PRECISION_DOUBLE ? 1 : 0};
        const int block = 256;
        const unsigned grid = (unsigned)((n + block - 1) / block);
        const int mode = edge_mode(c, walker_smem_bytes(block));
        const size_t smem = walker_smem_bytes(block) + (mode == EDGES_SHARED ? edges_smem_bytes(c) : 0);
        if (mode == EDGES_ARITH) trace_kernel<EDGES_ARITH><<<grid, block, smem, c->stream>>>(P);
        else if (mode == EDGES_SHARED) {
            if (smem > 48 * 1024) e = cudaFuncSetAttribute(trace_kernel<EDGES_SHARED>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e == cudaSuccess) trace_kernel<EDGES_SHARED><<<grid, block, smem, c->stream>>>(P);
        } else
            trace_kernel<EDGES_GLOBAL><<<grid, block, smem, c->stream>>>(P);
        c->launches += 1;
        if (e == cudaSuccess) e = cudaGetLastError();
    }
    if (e == cudaSuccess && d_nseg) e = cudaMemcpyAsync(nseg, d_nseg, (size_t)n * 4, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess && d_hash) e = cudaMemcpyAsync(hash, d_hash, (size_t)n * 8, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess && d_cells) e = cudaMemcpyAsync(cells, d_cells, (size_t)n * cap * 4, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess && d_lens) e = cudaMemcpyAsync(lens, d_lens, (size_t)n * cap * 8, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cleanup();
    if (e != cudaSuccess) return c->fail_cuda(e, "mr_trace_rays");
    return MR_OK;
}

}  // extern "C"

namespace {

template <typename Real, typename Rec, int MODE, bool TRACE>
int launch_ne_m(mr_ctx *c, const NextEventParams &P, int ndet_launch, int block, size_t smem)
{
    const long long gx = (P.n + block - 1) / block;
    if (gx > 0x7fffffffLL) return c->fail(MR_ERR_UNSUPPORTED, "batch too large for one launch");
    if (int rc = set_smem(c, next_event_kernel<Real, Rec, MODE, TRACE>, smem)) return rc;
    next_event_kernel<Real, Rec, MODE, TRACE><<<dim3((unsigned)gx, (unsigned)ndet_launch), block, smem, c->work_stream()>>>(P);
    c->launches += 1;
    MR_CUDA(c, cudaGetLastError());
    return MR_OK;
}

template <typename Real, typename Rec, bool TRACE>
int launch_ne_t(mr_ctx *c, const NextEventParams &P, int ndet_launch)
{
    const int block = c->block_threads;
    const size_t per_block = walker_smem_bytes(block) + (size_t)(c->M + c->N) * block * sizeof(Real);
    const int mode = edge_mode(c, per_block);
    const size_t smem = (mode == EDGES_SHARED ? edges_smem_bytes(c) : 0) + per_block;
    if (smem > 227 * 1024) return c->fail(MR_ERR_UNSUPPORTED, "materials x block threads exceed shared memory; lower MR_OPT_BLOCK_THREADS");
    switch (mode) {
    case EDGES_ARITH: return launch_ne_m<Real, Rec, EDGES_ARITH, TRACE>(c, P, ndet_launch, block, smem);
    case EDGES_SHARED: return launch_ne_m<Real, Rec, EDGES_SHARED, TRACE>(c, P, ndet_launch, block, smem);
    default: return launch_ne_m<Real, Rec, EDGES_GLOBAL, TRACE>(c, P, ndet_launch, block, smem);
    }
}

// next_event_tiled_kernel (mr_tiled.cuh): dictionary path with at most 16 distinct records
template <int MODE, bool TRACE>
int launch_ne_tiled_m(mr_ctx *c, const NextEventParams &P, const NextEventTiles &T, int ndet_launch, int block, size_t smem)
{
    const long long gx = (P.n + block - 1) / block;
    if (gx > 0x7fffffffLL) return c->fail(MR_ERR_UNSUPPORTED, "batch too large for one launch");
    if (int rc = set_smem(c, next_event_tiled_kernel<MODE, TRACE>, smem)) return rc;
    next_event_tiled_kernel<MODE, TRACE><<<dim3((unsigned)gx, (unsigned)ndet_launch), block, smem, c->work_stream()>>>(P, T);
    c->launches += 1;
    MR_CUDA(c, cudaGetLastError());
    return MR_OK;
}

template <bool TRACE>
int launch_ne_tiled(mr_ctx *c, const NextEventParams &P, int ndet_launch)
{
    const NextEventTiles T{c->d_dict, c->d_tiles, c->ndict, c->ntx, c->nty};
    const int block = c->block_threads;
    const size_t per_block = walker_smem_bytes(block) + (((size_t)(c->M + c->N) * block * sizeof(float) + 15) & ~(size_t)15) +
                             (size_t)kPerEntryMax * block * sizeof(float) + (size_t)c->ndict * sizeof(uint4);
    const int mode = edge_mode(c, per_block);
    const size_t smem = (mode == EDGES_SHARED ? edges_smem_bytes(c) : 0) + per_block;
    if (smem > 227 * 1024) return c->fail(MR_ERR_UNSUPPORTED, "materials x block threads exceed shared memory; lower MR_OPT_BLOCK_THREADS");
    switch (mode) {
    case EDGES_ARITH: return launch_ne_tiled_m<EDGES_ARITH, TRACE>(c, P, T, ndet_launch, block, smem);
    case EDGES_SHARED: return launch_ne_tiled_m<EDGES_SHARED, TRACE>(c, P, T, ndet_launch, block, smem);
    default: return launch_ne_tiled_m<EDGES_GLOBAL, TRACE>(c, P, T, ndet_launch, block, smem);
    }
}

template <bool TRACE>
int launch_next_event(mr_ctx *c, const NextEventParams &P, int ndet_launch)
{
    // (K = 1 meshes keep their 8-byte records: measured on config 2, 2.46 ms against 2.93 ms with the index tiles)
    if (record_path(c) == MR_PATH_TILED4 && c->layout != LAYOUT_K1) return launch_ne_tiled<TRACE>(c, P, ndet_launch);
    if (c->precision == MR_PRECISION_DOUBLE)
        return c->layout == LAYOUT_DK3 ? launch_ne_t<double, CellRec<LAYOUT_DK3>, TRACE>(c, P, ndet_launch)
                                       : launch_ne_t<double, CellRecGeneric<double>, TRACE>(c, P, ndet_launch);
    switch (c->layout) {
    case LAYOUT_K1: return launch_ne_t<float, CellRec<LAYOUT_K1>, TRACE>(c, P, ndet_launch);
    case LAYOUT_K2: return c->pair_records ? launch_ne_t<float, CellRec<LAYOUT_K2P>, TRACE>(c, P, ndet_launch) : launch_ne_t<float, CellRec<LAYOUT_K2>, TRACE>(c, P, ndet_launch);
    case LAYOUT_K3: return c->pair_records ? launch_ne_t<float, CellRec<LAYOUT_K3P>, TRACE>(c, P, ndet_launch) : launch_ne_t<float, CellRec<LAYOUT_K3>, TRACE>(c, P, ndet_launch);
    case LAYOUT_K4: return launch_ne_t<float, CellRec<LAYOUT_K4>, TRACE>(c, P, ndet_launch);
    case LAYOUT_D8: return launch_ne_t<float, CellRec<LAYOUT_D8>, TRACE>(c, P, ndet_launch);
    default: return launch_ne_t<float, CellRecGeneric<float>, TRACE>(c, P, ndet_launch);
    }
}

NextEventParams ne_params(mr_ctx *c, long long n, const void *d_rays)
{
    NextEventParams P{};
    P.mesh = mesh_dev(c);
    P.recs = c->d_recs;
    P.ids = c->d_ids;
    P.K = c->K;
    P.M = c->M;
    P.xs = c->d_xs;
    P.N = c->N;
    P.mix_off = c->d_mix_off;
    P.mix_nuc = c->d_mix_nuc;
    P.mix_w = c->d_mix_w;
    P.rays = d_rays;
    P.n = n;
    P.det = c->d_det;
    return P;
}

RzNextEventParams rz_ne_params(mr_ctx *c, long long n, const void *d_rays, int det_first, int ndet, double *det_sum,
                               unsigned long long *counters)
{
    RzNextEventParams Q{};
    Q.c.mesh = mesh_dev(c);
    Q.c.recs = c->d_recs;
    Q.c.ids = c->d_ids;
    Q.c.K = c->K;
    Q.c.M = c->M;
    Q.c.xs = c->d_xs;
    Q.c.N = c->N;
    Q.c.mix_off = c->d_mix_off;
    Q.c.mix_nuc = c->d_mix_nuc;
    Q.c.mix_w = c->d_mix_w;
    Q.c.rays = d_rays;
    Q.c.n = n;
    Q.c.counters = counters;
    Q.det = c->d_det;
    Q.det_first = det_first;
    Q.ndet = ndet;
    Q.det_sum = det_sum;
    return Q;
}

// all detectors against n device-resident events (grid.y = detectors, at most 65535 per launch)
int next_event_device(mr_ctx *c, long long n, const void *d_rays)
{
    NextEventParams P = ne_params(c, n, d_rays);
    P.det_sum = c->d_det_sum;
    P.counters = c->d_counters + 4;
    if (c->kev_used + 2 > c->kev.size()) {
        cudaEvent_t a = nullptr, b = nullptr;
        MR_CUDA(c, cudaEventCreate(&a));
        MR_CUDA(c, cudaEventCreate(&b));
        c->kev.push_back(a);
        c->kev.push_back(b);
    }
    MR_CUDA(c, cudaEventRecord(c->kev[c->kev_used], c->work_stream()));
    if (c->mesh_rz) {      // R-Z / spherical mesh: one persistent launch over all (event, detector) pairs, no ordering pre-pass
        if (int rc = launch_rz_next_event<false>(c, rz_ne_params(c, n, d_rays, 0, c->ndet, c->d_det_sum, c->d_counters + 4))) return rc;
        MR_CUDA(c, cudaEventRecord(c->kev[c->kev_used + 1], c->work_stream()));
        c->kev_used += 2;
        return MR_OK;
    }
    // detectors in groups whose ordering scratch stays below 2^25 (event, detector) pairs
    const int group = (int)std::max<long long>(1, std::min<long long>(c->ndet, (1LL << 25) / std::max<long long>(n, 1)));
    for (int first = 0; first < c->ndet; first += group) {
        const int count = std::min(group, c->ndet - first);
        P.det_first = first;
        if (int rc = order_rays(c, n, d_rays, &P.perm, count, first)) return rc;
        if (int rc = launch_next_event<false>(c, P, count)) return rc;
    }
    MR_CUDA(c, cudaEventRecord(c->kev[c->kev_used + 1], c->work_stream()));
    c->kev_used += 2;
    return MR_OK;
}

}  // namespace

extern "C" {

int mr_end_batch(mr_ctx *c)
{
    MR_ENTER(c);
    if (!c->d_tally) return c->fail(MR_ERR_STATE, "no mesh loaded");
    if (!c->d_prev) {
        c->d_prev = (double *)c->dev_alloc(sizeof(double) * c->ncell);
        c->d_s2 = (double *)c->dev_alloc(sizeof(double) * c->ncell);
        if (!c->d_prev || !c->d_s2) {
            c->dev_free(c->d_prev);
            c->dev_free(c->d_s2);
            c->d_prev = c->d_s2 = nullptr;
            return c->fail(MR_ERR_OOM, "device allocation failed (batch moments)");
        }
        MR_CUDA(c, cudaMemsetAsync(c->d_prev, 0, sizeof(double) * c->ncell, c->stream));
        MR_CUDA(c, cudaMemsetAsync(c->d_s2, 0, sizeof(double) * c->ncell, c->stream));
    }
    MR_CUDA(c, flush_accumulators(c));
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    const long long want = (c->ncell / 2 + 255) / 256 + 1;
    const unsigned grid = (unsigned)std::min<long long>(want, (long long)sms * 8);
    fold_batch_kernel<<<grid, 256, 0, c->stream>>>(c->d_tally, c->d_prev, c->d_s2, c->ncell);
    c->launches += 1;
    MR_CUDA(c, cudaGetLastError());
    c->nbatch += 1;
    return MR_OK;
}

int mr_read_moments(mr_ctx *c, double *sum, double *sumsq, int64_t *nbatch)
{
    MR_ENTER(c);
    if (!c->d_tally) return c->fail(MR_ERR_STATE, "no mesh loaded");
    if (nbatch) *nbatch = c->nbatch;
    if (!c->d_prev) {
        MR_CUDA(c, cudaStreamSynchronize(c->stream));
        if (sum) std::memset(sum, 0, sizeof(double) * c->ncell);
        if (sumsq) std::memset(sumsq, 0, sizeof(double) * c->ncell);
        return MR_OK;
    }
    if (sum) MR_CUDA(c, cudaMemcpyAsync(sum, c->d_prev, sizeof(double) * c->ncell, cudaMemcpyDeviceToHost, c->stream));
    if (sumsq) MR_CUDA(c, cudaMemcpyAsync(sumsq, c->d_s2, sizeof(double) * c->ncell, cudaMemcpyDeviceToHost, c->stream));
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    return MR_OK;
}

int mr_read_mean_sigma(mr_ctx *c, double *mean, double *sigma, int64_t *nbatch)
{
    MR_ENTER(c);
    if (!c->d_tally) return c->fail(MR_ERR_STATE, "no mesh loaded");
    if (!c->d_prev || c->nbatch < 1) return c->fail(MR_ERR_STATE, "no closed batch (call mr_end_batch first)");
    if (nbatch) *nbatch = c->nbatch;
    double *d_mean = (double *)c->dev_alloc(sizeof(double) * c->ncell);
    double *d_sigma = (double *)c->dev_alloc(sizeof(double) * c->ncell);
    if (!d_mean || !d_sigma) {
        c->dev_free(d_mean);
        c->dev_free(d_sigma);
        return c->fail(MR_ERR_OOM, "device allocation failed (mean / sigma)");
    }
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    const unsigned grid = (unsigned)std::min<long long>((c->ncell + 255) / 256, (long long)sms * 8);
    mean_sigma_kernel<<<grid, 256, 0, c->stream>>>(c->d_prev, c->d_s2, d_mean, d_sigma, c->ncell, c->nbatch);
    c->launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && mean) e = cudaMemcpyAsync(mean, d_mean, sizeof(double) * c->ncell, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess && sigma) e = cudaMemcpyAsync(sigma, d_sigma, sizeof(double) * c->ncell, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    c->dev_free(d_mean);
    c->dev_free(d_sigma);
    if (e != cudaSuccess) return c->fail_cuda(e, "mr_read_mean_sigma");
    return MR_OK;
}

int mr_load_detectors(mr_ctx *c, int ndet, const double *xyz)
{
    MR_ENTER(c);
    if (ndet < 1 || !xyz) return c->fail(MR_ERR_INVALID_ARG, "detectors: bad count or NULL array");
    if (ndet > 65535) return c->fail(MR_ERR_UNSUPPORTED, "detectors: at most 65535 points");
    for (int i = 0; i < 3 * ndet; ++i)
        if (!std::isfinite(xyz[i])) return c->fail(MR_ERR_INVALID_ARG, "detectors: coordinates must be finite");
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    c->dev_free(c->d_det);
    c->dev_free(c->d_det_sum);
    c->ndet = 0;
    c->d_det = (double *)c->dev_alloc(sizeof(double) * 3 * ndet);
    c->d_det_sum = (double *)c->dev_alloc(sizeof(double) * ndet);
    if (!c->d_det || !c->d_det_sum) {
        c->dev_free(c->d_det);
        c->dev_free(c->d_det_sum);
        c->d_det = c->d_det_sum = nullptr;
        return c->fail(MR_ERR_OOM, "device allocation failed (detectors)");
    }
    MR_CUDA(c, cudaMemcpyAsync(c->d_det, xyz, sizeof(double) * 3 * ndet, cudaMemcpyHostToDevice, c->stream));
    MR_CUDA(c, cudaMemsetAsync(c->d_det_sum, 0, sizeof(double) * ndet, c->stream));
    MR_CUDA(c, cudaMemsetAsync(c->d_counters + 4, 0, 4 * sizeof(unsigned long long), c->stream));
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    c->ndet = ndet;
    return MR_OK;
}

int mr_cast_next_event(mr_ctx *c, int64_t n, const void *rays, int where)
{
    MR_ENTER(c);
    if (n < 0 || (n > 0 && !rays) || (where != MR_WHERE_HOST && where != MR_WHERE_DEVICE))
        return c->fail(MR_ERR_INVALID_ARG, "next_event: bad count, NULL buffer or unknown location");
    if (int rc = ready_to_cast(c)) return rc;
    if (!c->ndet) return c->fail(MR_ERR_STATE, "no detectors loaded");
    if (n == 0) return MR_OK;
    if (int rc = upload_xs_desc(c)) return rc;
    return run_batch(c, n, rays, where, [c](long long count, const void *d_rays) { return next_event_device(c, count, d_rays); });
}

int mr_read_detectors(mr_ctx *c, double *out)
{
    MR_ENTER(c);
    if (!out) return c->fail(MR_ERR_INVALID_ARG, "read_detectors: out is NULL");
    if (!c->ndet) return c->fail(MR_ERR_STATE, "no detectors loaded");
    MR_CUDA(c, cudaMemcpyAsync(out, c->d_det_sum, sizeof(double) * c->ndet, cudaMemcpyDeviceToHost, c->stream));
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    return MR_OK;
}

int mr_clear_detectors(mr_ctx *c)
{
    MR_ENTER(c);
    if (!c->ndet) return c->fail(MR_ERR_STATE, "no detectors loaded");
    MR_CUDA(c, cudaMemsetAsync(c->d_det_sum, 0, sizeof(double) * c->ndet, c->stream));
    MR_CUDA(c, cudaMemsetAsync(c->d_counters + 4, 0, 4 * sizeof(unsigned long long), c->stream));
    return MR_OK;
}

int mr_trace_next_event(mr_ctx *c, int64_t n, const void *rays, int where, int det, uint32_t *nseg, uint64_t *hash,
                        double *tau, double *score)
{
    MR_ENTER(c);
    if (n < 0 || (n > 0 && !rays) || (where != MR_WHERE_HOST && where != MR_WHERE_DEVICE))
        return c->fail(MR_ERR_INVALID_ARG, "trace_next_event: bad count, NULL buffer or unknown location");
    if (int rc = ready_to_cast(c)) return rc;
    if (!c->ndet) return c->fail(MR_ERR_STATE, "no detectors loaded");
    if (det < 0 || det >= c->ndet) return c->fail(MR_ERR_INVALID_ARG, "trace_next_event: detector index out of range");
    if (n == 0) return MR_OK;
    if (int rc = upload_xs_desc(c)) return rc;
    const size_t rb = c->ray_bytes();
    void *d_rays = nullptr;
    uint32_t *d_nseg = nullptr;
    unsigned long long *d_hash = nullptr;
    double *d_tau = nullptr, *d_score = nullptr;
    auto cleanup = [&]() {
        if (where == MR_WHERE_HOST) c->dev_free(d_rays);
        c->dev_free(d_nseg); c->dev_free(d_hash); c->dev_free(d_tau); c->dev_free(d_score);
    };
    bool ok = true;
    if (where == MR_WHERE_HOST) ok = ok && (d_rays = c->dev_alloc((size_t)n * rb));
    if (nseg) ok = ok && (d_nseg = (uint32_t *)c->dev_alloc((size_t)n * 4));
    if (hash) ok = ok && (d_hash = (unsigned long long *)c->dev_alloc((size_t)n * 8));
    if (tau) ok = ok && (d_tau = (double *)c->dev_alloc((size_t)n * 8));
    if (score) ok = ok && (d_score = (double *)c->dev_alloc((size_t)n * 8));
    if (!ok) {
        cleanup();
        return c->fail(MR_ERR_OOM, "device allocation failed (next-event trace buffers)");
    }
    cudaError_t e = cudaSuccess;
    if (where == MR_WHERE_HOST) e = cudaMemcpyAsync(d_rays, rays, (size_t)n * rb, cudaMemcpyHostToDevice, c->stream);
    else {
        if ((uintptr_t)rays & 15) { cleanup(); return c->fail(MR_ERR_INVALID_ARG, "trace_next_event: device ray buffer must be 16-byte aligned"); }
        d_rays = const_cast<void *>(rays);
    }
    int rc = MR_OK;
    if (e == cudaSuccess && c->mesh_rz) {
        RzNextEventParams Q = rz_ne_params(c, n, d_rays, det, 1, nullptr, nullptr);
        Q.nseg = d_nseg; Q.hash = d_hash; Q.tau = d_tau; Q.score = d_score;
        rc = launch_rz_next_event<true>(c, Q);
    } else if (e == cudaSuccess) {
        NextEventParams P = ne_params(c, n, d_rays);
        P.det_first = det;
        P.nseg = d_nseg; P.hash = d_hash; P.tau = d_tau; P.score = d_score;
        rc = launch_next_event<true>(c, P, 1);
    }
    if (rc == MR_OK) {
        if (e == cudaSuccess && d_nseg) e = cudaMemcpyAsync(nseg, d_nseg, (size_t)n * 4, cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess && d_hash) e = cudaMemcpyAsync(hash, d_hash, (size_t)n * 8, cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess && d_tau) e = cudaMemcpyAsync(tau, d_tau, (size_t)n * 8, cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess && d_score) e = cudaMemcpyAsync(score, d_score, (size_t)n * 8, cudaMemcpyDeviceToHost, c->stream);
    }
    cudaError_t e2 = cudaStreamSynchronize(c->stream);
    if (e == cudaSuccess) e = e2;
    cleanup();
    if (rc != MR_OK) return rc;
    if (e != cudaSuccess) return c->fail_cuda(e, "mr_trace_next_event");
    return MR_OK;
}

}  // extern "C"

namespace {

void ring_free(mr_ctx *c)
{
    Ring *r = c->ring;
    if (!r) return;
    for (RingSlot *s : r->slots) {
        if (s->ev_copied) { cudaEventSynchronize(s->ev_copied); cudaEventDestroy(s->ev_copied); }
        if (s->ev_done) { cudaEventSynchronize(s->ev_done); cudaEventDestroy(s->ev_done); }
        if (s->pinned) cudaFreeHost(s->pinned);
        delete s;
    }
    if (r->ev_cast) cudaEventDestroy(r->ev_cast);
    c->dev_free(r->d_all);
    delete r;
    c->ring = nullptr;
}

// With r->ship_m held and the device current: ONE cast (one ordering pre-pass, one launch) over the rays of all pending slots.
int ring_cast_pending(mr_ctx *c, std::string *msg)
{
    Ring *r = c->ring;
    if (r->pend_n == 0) return MR_OK;
    const int first = r->pend_first, n = r->pend_n;
    const long long rays = r->pend_rays;
    r->pend_n = 0;
    r->pend_rays = 0;
    r->pend_full = true;
    c->kev_used = 0;
    const int rc = cast_device(c, rays, r->slots[first]->d_buf);
    if (rc != MR_OK) {
        *msg = c->err;
        return rc;
    }
    cudaError_t e = cudaSuccess;
    for (int i = first; i < first + n && e == cudaSuccess; ++i) e = cudaEventRecord(r->slots[i]->ev_done, c->stream);
    if (e == cudaSuccess) e = cudaEventRecord(r->ev_cast, c->stream);
    if (e != cudaSuccess) {
        *msg = std::string("CUDA error while casting ring buffers: ") + cudaGetErrorString(e);
        return MR_ERR_CUDA;
    }
    r->cast_recorded = true;
    r->casts += 1;
    return MR_OK;
}

// Hands slot s (count rays, all reserved) to the GPU.  Called by the thread that filled it, no ring lock held.
// The H2D copy is queued at once.  The cast is queued at once too unless an earlier cast of this ring is still running
// (MR_OPT_RING_MERGE auto): then the slot only joins the pending range, and the next ship that finds the GPU free -- or
// mr_ring_flush -- casts the whole range in one launch.  Ten 2^20-ray casts, each with its own pre-pass and its own ramp up
// and down, cost 7.4 ms of kernels on the PWR-like config where one 10^7-ray cast costs 6.0 + 0.3 ms.
void ring_ship(mr_ctx *c, RingSlot *s, long long count)
{
    Ring *r = c->ring;
    while (s->committed.load(std::memory_order_acquire) < count) std::this_thread::yield();   // other producers still copying in
    int rc = MR_OK;
    std::string msg;
    {
        std::lock_guard<std::mutex> g(r->ship_m);
        DeviceGuard guard(c->device);
        const size_t bytes = (size_t)count * c->ray_bytes();
        // a slot that does not extend the pending range (the ring wrapped, slots shipped out of order, a partial slot is
        // waiting) sends the range off first; this also puts ev_done of a pending slot behind its cast before the slot's
        // device buffer is written again
        if (r->pend_n > 0 && !(r->pend_full && s->index == r->pend_first + r->pend_n)) rc = ring_cast_pending(c, &msg);
        if (rc == MR_OK) {
            // is a cast of this ring still running?  (asked before this slot's copy is queued behind it)
            bool busy = c->ring_merge == 2;
            if (c->ring_merge == 1 && r->cast_recorded) {
                busy = cudaEventQuery(r->ev_cast) == cudaErrorNotReady;
                cudaGetLastError();
            }
            cudaError_t e = cudaStreamWaitEvent(c->copy_stream, s->ev_done, 0);
            if (e == cudaSuccess) e = cudaMemcpyAsync(s->d_buf, s->pinned, bytes, cudaMemcpyHostToDevice, c->copy_stream);
            if (e == cudaSuccess) e = cudaEventRecord(s->ev_copied, c->copy_stream);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(c->stream, s->ev_copied, 0);
            if (e != cudaSuccess) {
                rc = MR_ERR_CUDA;
                msg = std::string("CUDA error while shipping a ring buffer: ") + cudaGetErrorString(e);
            } else {
                if (r->pend_n == 0) r->pend_first = s->index;
                r->pend_n += 1;
                r->pend_rays += count;
                if (count < r->cap) r->pend_full = false;
                // auto: at most half the ring waits.  A waiting buffer's device half is only free again after the merged cast, and
                // the copy of the buffer that comes round to it next waits for that: with 4 buffers of 2^20 rays and unlimited
                // merging the producers stood still for 2.7 ms of a 12.4 ms step (10.7 ms without merging)
                const bool enough = c->ring_merge == 1 && r->pend_n >= std::max<int>(1, (int)r->slots.size() / 2);
                if (!busy || !r->pend_full || enough) rc = ring_cast_pending(c, &msg);
            }
        }
    }
    std::lock_guard<std::mutex> g(r->m);
    if (rc != MR_OK && r->error == MR_OK) { r->error = rc; r->error_msg = msg; }
    r->slots_shipped += 1;
    s->state = RingSlot::IN_FLIGHT;
    r->cv.notify_all();
}

// With r->m held: make r->open a slot that can take rays (waits for its last H2D copy if it is still in flight).
// r->open may move while this thread sleeps on the condition variable, so it is re-read after every wait.
void ring_acquire_open(mr_ctx *c, std::unique_lock<std::mutex> &lk)
{
    Ring *r = c->ring;
    if (r->slots[r->open]->state == RingSlot::FILLING) return;
    const auto t0 = std::chrono::steady_clock::now();
    bool waited = false;
    for (;;) {
        RingSlot *s = r->slots[r->open];
        if (s->state == RingSlot::FILLING) break;                 // another producer re-opened it meanwhile
        if (s->state == RingSlot::SHIPPING) {                     // its filler has not queued it yet
            waited = true;
            r->cv.wait(lk);
            continue;
        }
        if (s->state == RingSlot::IN_FLIGHT && cudaEventQuery(s->ev_copied) != cudaSuccess) {
            waited = true;
            cudaGetLastError();
            DeviceGuard guard(c->device);
            cudaEventSynchronize(s->ev_copied);     // every slot is in flight: the producers have to wait (lock held on purpose)
        }
        s->state = RingSlot::FILLING;
        s->cursor = 0;
        s->committed.store(0, std::memory_order_release);
        break;
    }
    if (waited) r->wait_ms += std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
}

}  // namespace

extern "C" {

int mr_ring_open(mr_ctx *c, int slots, int64_t rays_per_slot)
{
    MR_ENTER(c);
    if (c->ring) return c->fail(MR_ERR_STATE, "ring already open");
    if (slots < 2 || slots > 16 || rays_per_slot < 1024 || rays_per_slot > (1LL << 28))
        return c->fail(MR_ERR_INVALID_ARG, "ring: 2..16 slots of 1024..2^28 rays");
    if (int rc = ready_to_cast(c)) return rc;
    if (int rc = upload_xs_desc(c)) return rc;
    Ring *r = new Ring();
    c->ring = r;
    r->cap = rays_per_slot;
    const size_t bytes = (size_t)rays_per_slot * c->ray_bytes();
    // one device allocation behind all slots: consecutive slots can be cast as one batch (ring_ship)
    r->d_all = c->dev_alloc(bytes * (size_t)slots);
    if (!r->d_all || cudaEventCreateWithFlags(&r->ev_cast, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        ring_free(c);
        return c->fail(MR_ERR_OOM, "ring: device allocation failed");
    }
    for (int i = 0; i < slots; ++i) {
        RingSlot *s = new RingSlot();
        r->slots.push_back(s);
        s->index = i;
        s->d_buf = (char *)r->d_all + bytes * (size_t)i;
        bool ok = cudaMallocHost(&s->pinned, bytes) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&s->ev_copied, cudaEventDisableTiming) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&s->ev_done, cudaEventDisableTiming) == cudaSuccess;
        if (!ok) {
            cudaGetLastError();
            ring_free(c);
            return c->fail(MR_ERR_OOM, "ring: page-locked or device allocation failed");
        }
    }
    // grow the ordering scratch now: cast_device must not synchronise the stream while producers run
    // (for as many rays as a merged cast can hold: all slots)
    const long long most = c->ring_merge ? rays_per_slot * slots : rays_per_slot;
    if (c->sort_rays && most >= kSortMinRays) {
        const uint32_t *perm = nullptr;
        MR_CUDA(c, cudaMemsetAsync(r->d_all, 0, (size_t)most * c->ray_bytes(), c->stream));
        if (int rc = order_rays(c, most, r->d_all, &perm)) { ring_free(c); return rc; }
        MR_CUDA(c, cudaStreamSynchronize(c->stream));
    }
    return MR_OK;
}

int mr_ring_push(mr_ctx *c, int64_t n, const void *rays)
{
    if (!c) return MR_ERR_INVALID_ARG;
    Ring *r = c->ring;
    if (!r) return MR_ERR_STATE;
    if (n < 0 || (n > 0 && !rays)) return MR_ERR_INVALID_ARG;
    const size_t rb = c->ray_bytes();
    const char *src = (const char *)rays;
    while (n > 0) {
        RingSlot *s;
        long long off, take;
        bool full;
        {
            std::unique_lock<std::mutex> lk(r->m);
            if (r->error != MR_OK) return r->error;
            ring_acquire_open(c, lk);
            s = r->slots[r->open];
            off = s->cursor;
            take = std::min<long long>(n, r->cap - off);
            s->cursor += take;
            full = s->cursor == r->cap;
            if (full) {
                s->state = RingSlot::SHIPPING;
                r->open = (r->open + 1) % (int)r->slots.size();
            }
            r->rays_pushed += take;
        }
        std::memcpy((char *)s->pinned + (size_t)off * rb, src, (size_t)take * rb);
        s->committed.fetch_add(take, std::memory_order_acq_rel);
        if (full) ring_ship(c, s, r->cap);
        src += (size_t)take * rb;
        n -= take;
    }
    return MR_OK;
}

int mr_ring_flush(mr_ctx *c)
{
    if (!c) return MR_ERR_INVALID_ARG;
    Ring *r = c->ring;
    if (!r) return MR_ERR_STATE;
    RingSlot *s = nullptr;
    long long count = 0;
    {
        std::unique_lock<std::mutex> lk(r->m);
        RingSlot *o = r->slots[r->open];
        if (o->state == RingSlot::FILLING && o->cursor > 0) {
            s = o;
            count = o->cursor;
            o->state = RingSlot::SHIPPING;
            r->open = (r->open + 1) % (int)r->slots.size();
        }
    }
    if (s) ring_ship(c, s, count);
    std::unique_lock<std::mutex> lk(r->m);
    while (true) {   // every slot a producer marked SHIPPING has been queued
        bool pending = false;
        for (RingSlot *q : r->slots) pending = pending || q->state == RingSlot::SHIPPING;
        if (!pending) break;
        r->cv.wait(lk);
    }
    lk.unlock();
    {   // slots held back for a merged cast go now
        std::lock_guard<std::mutex> g(r->ship_m);
        DeviceGuard guard(c->device);
        std::string msg;
        const int rc = ring_cast_pending(c, &msg);
        if (rc != MR_OK) {
            std::lock_guard<std::mutex> g2(r->m);
            if (r->error == MR_OK) { r->error = rc; r->error_msg = msg; }
        }
    }
    lk.lock();
    if (r->error != MR_OK) {
        c->err = r->error_msg;
        return r->error;
    }
    return MR_OK;
}

// Measurement aid for the producer ring: `producers` threads INSIDE the library push the host batch through mr_ring_push
// in pieces of `rays_per_push` rays (thread k owns the k-th contiguous share), then the ring is flushed.  A producer written in
// Python measures the interpreter, not the ring.  dry_run != 0: the threads copy the same pieces into private scratch buffers
// instead (what the producers cost with no ring and no GPU behind them).
int mr_ring_bench_producers(mr_ctx *c, int64_t n, const void *rays, int producers, int64_t rays_per_push, int dry_run, double *wall_ms)
{
    MR_ENTER(c);
    if (n < 0 || (n > 0 && !rays) || producers < 1 || producers > 256 || rays_per_push < 1)
        return c->fail(MR_ERR_INVALID_ARG, "ring_bench_producers: bad count, NULL buffer, or producers / rays_per_push out of range");
    if (!dry_run && !c->ring) return c->fail(MR_ERR_STATE, "ring_bench_producers: no producer ring is open");
    const size_t rb = c->ray_bytes();
    std::atomic<int> rc{MR_OK};
    std::atomic<bool> stop{false};      // one producer's failed push ends the others' loops too
    // dry run: every thread's whole share goes to a private buffer of its own size (destination lines not in cache, as in the
    // ring), allocated and touched before the clock starts
    std::vector<std::unique_ptr<char[]>> scratches((size_t)producers);
    if (dry_run)
        for (int k = 0; k < producers; ++k) {
            const size_t bytes = (size_t)std::max<int64_t>(n * (k + 1) / producers - n * k / producers, 1) * rb;
            scratches[(size_t)k].reset(new char[bytes]);
            std::memset(scratches[(size_t)k].get(), 0, bytes);
        }
    const auto t0 = std::chrono::steady_clock::now();
    std::vector<std::thread> pool;
    for (int k = 0; k < producers; ++k) {
        const int64_t lo = n * k / producers, hi = n * (k + 1) / producers;
        char *const scratch_k = scratches[(size_t)k].get();
        pool.emplace_back([=, &rc, &stop]() {
            struct { char *p; char *get() const { return p; } } scratch{scratch_k};
            for (int64_t i = lo; i < hi && !stop.load(std::memory_order_relaxed); i += rays_per_push) {
                const int64_t m = std::min<int64_t>(rays_per_push, hi - i);
                const char *src = (const char *)rays + (size_t)i * rb;
                if (dry_run) {
                    std::memcpy(scratch.get() + (size_t)(i - lo) * rb, src, (size_t)m * rb);
                    asm volatile("" ::"r"(scratch.get()) : "memory");
                } else {
                    const int r = mr_ring_push(c, m, src);
                    if (r != MR_OK) { rc.store(r); stop.store(true); return; }
                }
            }
        });
    }
    for (std::thread &t : pool) t.join();
    int ret = rc.load();
    if (!dry_run) {     // also after a failed push: what the other producers had put into open slots is shipped, no slot stays half filled
        const int flushed = mr_ring_flush(c);
        if (ret == MR_OK) ret = flushed;
    }
    if (wall_ms) *wall_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    return ret;
}

int mr_ring_close(mr_ctx *c)
{
    if (!c) return MR_ERR_INVALID_ARG;
    if (!c->ring) return MR_OK;
    const int rc = mr_ring_flush(c);
    DeviceGuard guard(c->device);
    cudaStreamSynchronize(c->copy_stream);
    cudaStreamSynchronize(c->stream);
    ring_free(c);
    return rc;
}

int mr_ring_get_stats(mr_ctx *c, mr_ring_stats *out)
{
    if (!c || !out) return MR_ERR_INVALID_ARG;
    std::memset(out, 0, sizeof(*out));
    Ring *r = c->ring;
    if (!r) return MR_ERR_STATE;
    {
        std::lock_guard<std::mutex> g(r->m);
        out->rays_pushed = r->rays_pushed;
        out->slots_shipped = r->slots_shipped;
        out->producer_wait_ms = r->wait_ms;
    }
    std::lock_guard<std::mutex> g2(r->ship_m);     // (never taken while r->m is held: ring_ship and mr_ring_flush nest them the other way)
    out->casts = r->casts;
    return MR_OK;
}

int mr_set_option(mr_ctx *c, int option, int64_t value)
{
    MR_ENTER(c);
    switch (option) {
    case MR_OPT_BLOCK_THREADS:
        if (value < 32 || value > 256 || (value & 31)) return c->fail(MR_ERR_INVALID_ARG, "block threads must be a multiple of 32 in [32, 256]");
        c->block_threads = (int)value;
        return MR_OK;
    case MR_OPT_RZ_BLOCK_THREADS:
        if (value < 32 || value > 256 || (value & 31)) return c->fail(MR_ERR_INVALID_ARG, "block threads must be a multiple of 32 in [32, 256]");
        c->rz_block_threads = (int)value;
        return MR_OK;
    case MR_OPT_SORT_RAYS:
        if (value != 0 && value != 1) return c->fail(MR_ERR_INVALID_ARG, "sort option is 0 or 1");
        c->sort_rays = (int)value;
        return MR_OK;
    case MR_OPT_STAGE_RAYS:
        if (value < 1024 || value > (1LL << 26)) return c->fail(MR_ERR_INVALID_ARG, "staging chunk must be in [1024, 2^26] rays");
        c->stage_rays = value;
        return MR_OK;
    case MR_OPT_PAIR_RECORDS:
        if (value != 0 && value != 1) return c->fail(MR_ERR_INVALID_ARG, "pair-records option is 0 or 1");
        c->pair_records = (int)value;
        return MR_OK;
    case MR_OPT_AGGREGATE_FIRST:
        if (value < 0 || value > 1 << 20) return c->fail(MR_ERR_INVALID_ARG, "aggregate-first option is a segment count >= 0");
        c->agg_first = (int)value;
        return MR_OK;
    case MR_OPT_TILED_INDEX:
        if (value != 0 && value != 1) return c->fail(MR_ERR_INVALID_ARG, "tiled-index option is 0 or 1");
        c->tiled_opt = (int)value;
        return MR_OK;
    case MR_OPT_FUSED_TALLY:
        if (value < 0 || value > 2) return c->fail(MR_ERR_INVALID_ARG, "fused-tally option is 0 (off), 1 (on) or 2 (auto)");
        c->fused_opt = (int)value;
        return MR_OK;
    case MR_OPT_ORDER_MODE:
        if (value < 0 || value > 2) return c->fail(MR_ERR_INVALID_ARG, "order mode is 0 (auto), 1 (slab-major) or 2 (longest first)");
        c->order_mode = (int)value;
        return MR_OK;
    case MR_OPT_COPY_THREADS:
        if (value < 1 || value > 64) return c->fail(MR_ERR_INVALID_ARG, "copy threads must be in [1, 64]");
        c->copy_threads = (int)value;
        return MR_OK;
    case MR_OPT_COOP_FLUSH:
        if (value < 0 || value > 3) return c->fail(MR_ERR_INVALID_ARG, "cooperative-flush option is 0 (off), 1 (on), 2 (auto) or 3 (pairs by shuffle)");
        c->coop_opt = (int)value;
        return MR_OK;
    case MR_OPT_WHOLE_BATCH:
        if (value < 0 || value > 2) return c->fail(MR_ERR_INVALID_ARG, "whole-batch option is 0 (never), 1 (always) or 2 (auto)");
        c->whole_opt = (int)value;
        return MR_OK;
    case MR_OPT_RING_MERGE:
        if (value < 0 || value > 2) return c->fail(MR_ERR_INVALID_ARG, "ring-merge option is 0 (one cast per buffer), 1 (auto) or 2 (hold until flush)");
        MR_NO_RING(c, "ring-merge option");
        c->ring_merge = (int)value;
        return MR_OK;
    case MR_OPT_TILED_TALLY:
        if (value != 0 && value != 1) return c->fail(MR_ERR_INVALID_ARG, "tiled-tally option is 0 or 1");
        c->tiled_tally_opt = (int)value;
        return MR_OK;
    case MR_OPT_COARSE_RECORDS:
        if (value != 0 && value != 1) return c->fail(MR_ERR_INVALID_ARG, "coarse-records option is 0 or 1");
        c->coarse_opt = (int)value;
        return MR_OK;
    case MR_OPT_DEFER_POOL_ENTRIES:
        if (value < 0 || value > (1LL << 32)) return c->fail(MR_ERR_INVALID_ARG, "deferred-tally pool size is 0 (auto) or a number of pairs up to 2^32");
        MR_CUDA(c, cudaStreamSynchronize(c->stream));
        free_defer(c);
        c->defer_pool_fixed = value;
        return MR_OK;
    case MR_OPT_DEFER_REGION_SHIFT:
        if (value != 0 && (value < 8 || value > 30)) return c->fail(MR_ERR_INVALID_ARG, "deferred-tally region shift is 0 (auto) or in [8, 30]");
        MR_CUDA(c, cudaStreamSynchronize(c->stream));
        free_defer(c);
        c->defer_shift_fixed = (int)value;
        return MR_OK;
    case MR_OPT_DEFERRED_TALLY:
        if (value < 0 || value > 2) return c->fail(MR_ERR_INVALID_ARG, "deferred-tally option is 0 (off), 1 (on) or 2 (auto)");
        if (value == 1 && c->fused && c->fused_dirty) {
            MR_CUDA(c, flush_accumulators(c));
        }
        c->defer_opt = (int)value;
        return MR_OK;
    }
    return c->fail(MR_ERR_INVALID_ARG, "unknown option");
}

int mr_get_option(mr_ctx *c, int option, int64_t *value)
{
    MR_ENTER(c);
    if (!value) return c->fail(MR_ERR_INVALID_ARG, "value is NULL");
    switch (option) {
    case MR_OPT_BLOCK_THREADS: *value = c->block_threads; return MR_OK;
    case MR_OPT_SORT_RAYS: *value = c->sort_rays; return MR_OK;
    case MR_OPT_RZ_BLOCK_THREADS: *value = c->rz_block_threads; return MR_OK;
    case MR_OPT_STAGE_RAYS: *value = c->stage_rays; return MR_OK;
    case MR_OPT_COPY_THREADS: *value = c->copy_threads; return MR_OK;
    case MR_OPT_PAIR_RECORDS: *value = c->pair_records; return MR_OK;
    case MR_OPT_ORDER_MODE: *value = c->order_mode; return MR_OK;
    case MR_OPT_FUSED_TALLY: *value = c->fused_opt; return MR_OK;
    case MR_OPT_TILED_INDEX: *value = c->tiled_opt; return MR_OK;
    case MR_OPT_AGGREGATE_FIRST: *value = c->agg_first; return MR_OK;
    case MR_OPT_COARSE_RECORDS: *value = c->coarse_opt; return MR_OK;
    case MR_OPT_COOP_FLUSH: *value = c->coop_opt; return MR_OK;
    case MR_OPT_TILED_TALLY: *value = c->tiled_tally_opt; return MR_OK;
    case MR_OPT_WHOLE_BATCH: *value = c->whole_opt; return MR_OK;
    case MR_OPT_RING_MERGE: *value = c->ring_merge; return MR_OK;
    case MR_INFO_RECORD_PATH: *value = record_path(c); return MR_OK;
    case MR_INFO_DISTINCT_RECORDS: *value = c->ndict; return MR_OK;
    case MR_INFO_COARSE_SHIFT: *value = c->cshift; return MR_OK;
    case MR_OPT_DEFERRED_TALLY: *value = c->defer_opt; return MR_OK;
    case MR_OPT_DEFER_POOL_ENTRIES: *value = c->defer_pool_fixed; return MR_OK;
    case MR_OPT_DEFER_REGION_SHIFT: *value = c->defer_shift_fixed; return MR_OK;
    case MR_INFO_DEFERRED: *value = use_deferred(c, record_path(c)) ? 1 : 0; return MR_OK;
    case MR_INFO_DEFER_DIRECT_PAIRS: {
        unsigned long long v = 0;
        if (c->d_defer_ctl) {
            MR_CUDA(c, cudaMemcpyAsync(&v, c->d_defer_ctl + 66, 8, cudaMemcpyDeviceToHost, c->stream));
            MR_CUDA(c, cudaStreamSynchronize(c->stream));
        }
        *value = (int64_t)v;
        return MR_OK;
    }
    }
    return c->fail(MR_ERR_INVALID_ARG, "unknown option");
}

}  // extern "C"

// =================================================================================================
// Measurement aid: the L2 fp64-atomic ceiling (mr_microbench.cuh)
// =================================================================================================
extern "C" int mr_microbench_red(int device, int64_t ncell, int group, int gather_bytes, int64_t lane_ops, int reps,
                                 double *best_ms, double *mean_ms)
{
    if (ncell < 1024 || ncell > 0xffffffffLL || group < 1 || group > 32 || (group & (group - 1)) || lane_ops < 1 || reps < 1 ||
        (gather_bytes != 0 && gather_bytes != 16 && gather_bytes != 32) || !best_ms)
        return MR_ERR_INVALID_ARG;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) {
        cudaGetLastError();
        return MR_ERR_CUDA;
    }
    DeviceGuard guard(device);
    RedBenchParams P{};
    P.ncell = (unsigned)ncell;
    P.group = group;
    P.gather_bytes = gather_bytes;
    P.iters = 64;
    const long long threads = std::max<long long>(128, (lane_ops + P.iters - 1) / P.iters / 128 * 128);
    double *tally = nullptr;
    uint4 *recs = nullptr;
    unsigned *sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    auto done = [&](int code) {
        cudaFree(tally);
        cudaFree(recs);
        cudaFree(sink);
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
        cudaGetLastError();
        return code;
    };
    if (cudaMalloc(&tally, (size_t)ncell * 8) != cudaSuccess || cudaMalloc(&sink, 4) != cudaSuccess ||
        (gather_bytes && cudaMalloc(&recs, (size_t)ncell * gather_bytes) != cudaSuccess))
        return done(MR_ERR_OOM);
    cudaMemset(tally, 0, (size_t)ncell * 8);
    if (recs) cudaMemset(recs, 0, (size_t)ncell * gather_bytes);
    P.tally = tally;
    P.recs = recs;
    P.sink = sink;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return done(MR_ERR_CUDA);
    double best = 1e300, sum = 0.0;
    for (int r = -2; r < reps; ++r) {                       // two warm-up launches
        cudaEventRecord(e0, 0);
        red_bench_kernel<<<(unsigned)(threads / 128), 128>>>(P);
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) return done(MR_ERR_CUDA);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r >= 0) {
            best = std::min(best, (double)ms);
            sum += ms;
        }
    }
    *best_ms = best;
    if (mean_ms) *mean_ms = sum / reps;
    return done(MR_OK);
}

// ---- mr_cast_rays_static: the cast for callers that cannot allocate device memory ------------------------------
//
// mr_cast_rays orders a batch before it casts it (mr_sort.cuh), and the ordering pre-pass needs scratch in global
// memory -- a key and a sorted position per ray, a histogram of the keys -- which order_rays() allocates, and grows,
// on demand.  Some hosts cannot allow that inside their transport loop:
//   * a Monte Carlo code that claims the whole device for its own pool at start-up leaves nothing to allocate from;
//   * cudaMalloc / cudaFree wait for the device to go idle, which stalls the CPU/GPU overlap the method lives on
//      and can deadlock a thread that holds a lock another stream's callback wants;
//   * code under a fixed memory budget (several ranks sharing one GPU) must know its footprint before the run.
// For them the same pre-pass runs here out of ONE fixed array that is part of the library image.  The array is device
// memory of every GPU that loads libmonteray.so, from load to process exit, whether or not this entry point is used.
//
// Shared state: every context and every stream of a device use the same array, and a call leaves its keys and
// positions in it.  Only the histogram has to start at zero; it is cleared on the stream at the start of every call.
// Two calls whose GPU work overlaps in time (two contexts, or one context moved to another stream while the earlier
// call is still running) race on the array and corrupt each other's ray order.
constexpr int kStaticMaxKeys = 256 * 128 + 1;                     // order_rays(): <= 256 z-slabs x 128 length buckets + "rejected"
constexpr size_t kStaticHistWords = ((size_t)kStaticMaxKeys + 1 + 63) & ~(size_t)63;
constexpr size_t kStaticWords = 2 * (size_t)MR_STATIC_MAX_RAYS + kStaticHistWords;   // keys | positions | histogram

static __device__ __align__(256) uint32_t g_static_scratch[kStaticWords];           // 2.1 MB per GPU

namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
uint32_t *g_static_addr[kStaticMaxDevices] = {};

// Device address of g_static_scratch on the CURRENT device (the caller has made the context's device current).  In host
// code the name g_static_scratch is only a handle for the runtime, not a pointer a kernel could use: the address has
// to be asked for, once per device.
int static_scratch(mr_ctx *c, uint32_t **out)
{
    if (c->device < 0 || c->device >= kStaticMaxDevices) return c->fail(MR_ERR_UNSUPPORTED, "cast_rays_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_addr[c->device]) {
        void *p = nullptr;
        MR_CUDA(c, cudaGetSymbolAddress(&p, g_static_scratch));
        g_static_addr[c->device] = static_cast<uint32_t *>(p);
    }
    *out = g_static_addr[c->device];
    return MR_OK;
}

}  // namespace

extern "C" int mr_cast_rays_static(mr_ctx *c, int64_t n, const void *d_rays)
{
    MR_ENTER(c);
    if (n < 0 || (n > 0 && !d_rays)) return c->fail(MR_ERR_INVALID_ARG, "cast_rays_static: bad count or NULL buffer");
    if (n > MR_STATIC_MAX_RAYS)
        return c->fail(MR_ERR_INVALID_ARG, "cast_rays_static: " + std::to_string((long long)n) + " rays in one call, the fixed scratch holds " +
                                               std::to_string((long long)MR_STATIC_MAX_RAYS) + " (MR_STATIC_MAX_RAYS): split the batch");
    if ((uintptr_t)d_rays & 15) return c->fail(MR_ERR_INVALID_ARG, "cast_rays_static: device ray buffer must be 16-byte aligned");
    MR_NO_RING(c, "cast_rays_static");
    if (int rc = ready_to_cast(c)) return rc;
    const int path = record_path(c);
    if (path == MR_PATH_RZ) return c->fail(MR_ERR_UNSUPPORTED, "cast_rays_static: Cartesian meshes only");
    if (use_deferred(c, path))
        return c->fail(MR_ERR_UNSUPPORTED, "cast_rays_static: the deferred tally keeps a pool that is sized per batch; set MR_OPT_DEFERRED_TALLY to 0");
    if (c->xs_dirty) {
        // the table descriptors are re-sent after every table load; their device buffers are made by the first ordinary cast
        bool mixtures = false;
        for (int m = 0; m < c->M && m < (int)c->mix.size(); ++m) mixtures = mixtures || !c->mix[m].empty();
        if (!c->d_xs || (mixtures && !c->d_mix_off))
            return c->fail(MR_ERR_STATE, "cast_rays_static: set-up is not finished -- make one mr_cast_rays call (one ray is enough) after loading the tables");
        if (int rc = upload_xs_desc(c)) return rc;
    }
    if (n == 0) return MR_OK;
    uint32_t *scratch = nullptr;
    if (int rc = static_scratch(c, &scratch)) return rc;

    cudaStream_t ws = c->work_stream();
    c->kev_used = 0;            // no per-kernel events here (mr_stats.last_kernel_ms stays 0): growing that list allocates
    MR_CUDA(c, cudaEventRecord(c->ev_t0, ws));

    CastParams P{};
    P.mesh = mesh_dev(c);
    P.recs = c->d_recs;
    P.ids = c->d_ids;
    P.K = c->K;
    P.M = c->M;
    P.xs = c->d_xs;
    P.N = c->N;
    P.mix_off = c->d_mix_off;
    P.mix_nuc = c->d_mix_nuc;
    P.mix_w = c->d_mix_w;
    P.rays = d_rays;
    P.perm = nullptr;
    P.n = n;
    P.agg_first = c->agg_first;
    P.tally = c->d_tally;
    P.counters = c->d_counters;

    // the ordering pre-pass, as order_rays() decides it, in its global-atomic form (classify, scan, scatter): that form
    // needs no per-CTA histograms, so the scratch stays small
    if (c->sort_rays && n >= kSortMinRays && edges_smem_bytes(c) <= kEdgesSmemMax) {
        const int nlen = 128;
        const int zdiv = (c->nz + 255) / 256;
        const int nslab = (c->nz + zdiv - 1) / zdiv;
        const int maxlen = c->nx + c->ny + c->nz;
        int lshift = 0;
        while ((maxlen >> lshift) >= nlen) ++lshift;
        const int nkeys = nslab * nlen + 1;
        if (nkeys > kStaticMaxKeys) return c->fail(MR_ERR_UNSUPPORTED, "cast_rays_static: more ordering keys than the fixed scratch holds");
        uint32_t *d_keys = scratch, *d_perm = scratch + MR_STATIC_MAX_RAYS, *d_hist = scratch + 2 * (size_t)MR_STATIC_MAX_RAYS;
        SortParams S{mesh_dev(c), d_rays, (long long)n, c->precision == MR_PRECISION_DOUBLE ? 1 : 0,
                     zdiv, lshift, nlen, nkeys, d_keys, d_hist, d_perm, nullptr, 0,
                     c->order_mode == 2 || (c->order_mode == 0 && c->resident_bytes() <= c->l2_bytes / 2) ? 1 : 0, nslab,
                     c->mesh_arith ? 1 : 0, 0, nullptr};
        const size_t smem = edges_smem_bytes(c);
        MR_CUDA(c, cudaMemsetAsync(d_hist, 0, ((size_t)nkeys + 1) * 4, ws));     // the last call's prefix sums are still there
        const unsigned grid = (unsigned)((n + 255) / 256);
        if (int rc = set_smem(c, classify_kernel, smem)) return rc;
        classify_kernel<<<grid, 256, smem, ws>>>(S);
        scan_kernel<<<1, 1024, 0, ws>>>(d_hist, nkeys);
        scatter_kernel<<<grid, 256, 0, ws>>>(S);
        c->launches += 3;
        MR_CUDA(c, cudaGetLastError());
        P.perm = d_perm;
    }

    // the record paths of cast_device(), minus the two refused above
    int rc;
    switch (path) {
    case MR_PATH_DOUBLE_K3: rc = launch_cast_or_coop<double, CellRec<LAYOUT_DK3>>(c, P, true); break;
    case MR_PATH_DOUBLE_GENERIC: rc = launch_cast_t<double, CellRecGeneric<double>>(c, P); break;
    case MR_PATH_TILED4: case MR_PATH_TILED8: case MR_PATH_TILED16:
        P.dict = c->d_dict;
        P.tiles = c->d_tiles;
        P.ndict = c->ndict;
        P.ntx = c->ntx;
        P.nty = c->nty;
        if (c->tiled_tally_opt && c->d_tally_t && !c->tally_borrowed) {
            P.tally_t = c->d_tally_t;
            rc = c->tile_bits == 4 ? launch_tiled<4>(c, P) : c->tile_bits == 8 ? launch_tiled<8>(c, P) : launch_tiled<16>(c, P);
        } else
            rc = c->tile_bits == 4 ? launch_cast_or_coop<float, TiledRec<4>>(c, P)
               : c->tile_bits == 8 ? launch_cast_or_coop<float, TiledRec<8>>(c, P) : launch_cast_or_coop<float, TiledRec<16>>(c, P);
        break;
    case MR_PATH_COARSE:
        P.crecs = c->d_crecs;
        P.cshift = c->cshift;
        P.cnx = c->cnx;
        P.cny = c->cny;
        rc = launch_cast_t<float, CellRec<LAYOUT_C4>>(c, P);
        break;
    case MR_PATH_K1: rc = launch_cast_or_coop<float, CellRec<LAYOUT_K1>>(c, P); break;
    case MR_PATH_K2: rc = launch_cast_t<float, CellRec<LAYOUT_K2>>(c, P); break;
    case MR_PATH_K3: rc = launch_cast_t<float, CellRec<LAYOUT_K3>>(c, P); break;
    case MR_PATH_K2_PAIRS: rc = launch_cast_t<float, CellRec<LAYOUT_K2P>>(c, P); break;
    case MR_PATH_K3_PAIRS: rc = launch_cast_or_coop<float, CellRec<LAYOUT_K3P>>(c, P, true); break;
    case MR_PATH_K4_FUSED: rc = launch_cast_t<float, CellRec<LAYOUT_K4F>>(c, P); c->fused_dirty = true; break;
    case MR_PATH_K4: rc = launch_cast_t<float, CellRec<LAYOUT_K4>>(c, P); break;
    case MR_PATH_DENSE8: rc = launch_cast_or_coop<float, CellRec<LAYOUT_D8>>(c, P); break;
    default: rc = launch_cast_t<float, CellRecGeneric<float>>(c, P);
    }
    if (rc) return rc;
    MR_CUDA(c, cudaEventRecord(c->ev_t1, ws));
    c->have_timing = true;
    return MR_OK;
}
