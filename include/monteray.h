/*
 * monteray.h -- C ABI of the B200-native VRC (volumetric-ray-casting) fluence-tally library.
 *
 * The library is the GPU side of the method of arXiv:1706.07476 (PAPER.md = the paper's text):
 * a host Monte Carlo random walk fills a buffer with rays (one per sampled outgoing
 * direction/energy at a collision or source event) and hands the full buffer to
 * the library (Fig. 4); for every ray the GPU evaluates all cross sections at
 * the ray's energy, casts the ray through the whole 3-D Cartesian mesh and scores Eq. (4)
 * into every crossed cell (Fig. 5); the tally stays on the GPU until it is read
 * back at the end.
 *
 * Conventions that hold for every call:
 *   - plain C, no exceptions cross the boundary; every function returns an mr_status;
 *     mr_last_error(ctx) gives a human-readable message owned by the context.
 *   - "host" pointers are ordinary CPU memory (pageable or pinned); "device" pointers are
 *     CUDA device memory on the context's device.  The caller owns every array it passes.
 *     The library has copied (or consumed) a HOST input before the call returns, so the
 *     caller may free or overwrite it at once -- the paper's "the CPU cleared the buffer and
 *     resumed".  A DEVICE input of mr_cast_rays / mr_trace_rays is read by
 *     work queued on the context's stream: keep it alive and unmodified until that work
 *     has finished (stream order, or mr_sync).
 *   - outputs are caller-allocated host arrays.
 *   - one context is used by one host thread at a time.  All device work of a context is
 *     ordered on ONE CUDA stream (mr_set_stream; default: the legacy default stream): the
 *     library's internal copy and compute streams fork from it and join it again before a
 *     call returns, so work the caller queues on that stream afterwards sees the results.
 *   - cell linear index c = ix + nx*(iy + ny*iz), x fastest.
 *   - units: cm, MeV, g/cc, cm^2/g; the tally is raw weight*cm sums (no volume or source
 *     normalisation: that is host-side bookkeeping, off the hot path).
 * Readings of the paper where it is silent (Q1..Q20) are listed in DESIGN.md §3.
 */
#ifndef MONTERAY_H
#define MONTERAY_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define MR_API __attribute__((visibility("default")))
#else
#define MR_API
#endif

typedef struct mr_ctx mr_ctx;

typedef enum {
    MR_OK = 0,
    MR_ERR_INVALID_ARG = 1, /* bad pointer/size/value; the context is unchanged */
    MR_ERR_STATE = 2,       /* wrong call order (e.g. cast before all tables are loaded) */
    MR_ERR_CUDA = 3,        /* a CUDA call failed; sticky errors keep being reported */
    MR_ERR_OOM = 4,         /* device or pinned-host allocation failed */
    MR_ERR_UNSUPPORTED = 5  /* a size beyond MR_MAX_* */
} mr_status;

/* Precision mode ("double-precision operations ... but using single precision
 * cross-sections and distances"; reading Q1):
 *   MIXED : fp32 energy grids, sigma tables, ray records and cell coefficients; fp64 mesh
 *           traversal, Eq. (4) evaluation and tally.  Ray record = 8 floats (32 B).
 *   DOUBLE: everything fp64.  Ray record = 8 doubles (64 B). */
enum { MR_PRECISION_MIXED = 0, MR_PRECISION_DOUBLE = 1 };

/* Where a ray buffer lives. */
enum { MR_WHERE_HOST = 0, MR_WHERE_DEVICE = 1 };

#define MR_MAX_MATERIALS 64
#define MR_MAX_SLOTS 16
#define MR_MAX_NUCLIDES 64
#define MR_MAX_MIX 16
#define MR_STATIC_MAX_RAYS 262144 /* most rays one mr_cast_rays_static call takes (2^18) */

/* Optional device-memory allocator supplied by the caller (the Python binding passes one that
 * hands out torch caching-allocator blocks).  alloc returns a device pointer aligned to 256 B
 * or NULL; both are called on the thread that calls into the library. */
typedef void *(*mr_alloc_fn)(void *user, size_t bytes, int device);
typedef void (*mr_free_fn)(void *user, void *ptr, int device);
typedef struct {
    mr_alloc_fn alloc;
    mr_free_fn free;
    void *user;
} mr_allocator;

typedef struct {
    int64_t rays_accepted;  /* rays cast since creation or the last mr_clear_tally */
    int64_t rays_rejected;  /* rays refused by the validation rule below */
    int64_t segments;       /* ray-cell segments scored (zero-length ones included) */
    int64_t kernel_launches;/* kernels this context has launched since creation */
    double last_cast_ms;    /* device time of the most recent mr_cast_rays work (copies and all kernels) */
    double last_kernel_ms;  /* device time of the cast kernel alone in that call (summed over its chunks) */
    int64_t ne_pairs_accepted; /* next-event: (event, detector) pairs scored since mr_load_detectors / mr_clear_detectors */
    int64_t ne_pairs_rejected; /* next-event: pairs refused by the rule of mr_cast_next_event */
    int64_t ne_segments;       /* next-event: cells crossed between events and detectors */
} mr_stats;

/* ---- life cycle -------------------------------------------------------------------------- */

/* Creates a context on CUDA device `device`.  `alloc` may be NULL (cudaMalloc is used).
 * Errors: INVALID_ARG (out NULL, unknown precision, bad device), CUDA. */
MR_API int mr_create(mr_ctx **out, int device, int precision);
MR_API int mr_create_ex(mr_ctx **out, int device, int precision, const mr_allocator *alloc);

/* Synchronises the stream, frees every device and pinned buffer.  NULL is accepted. */
MR_API int mr_destroy(mr_ctx *ctx);

/* Makes `cuda_stream` (a cudaStream_t passed as void*, NULL = legacy default stream) the
 * stream all later work of this context is queued on.  Pending work is synchronised first. */
MR_API int mr_set_stream(mr_ctx *ctx, void *cuda_stream);

/* Message of the last error of this context ("" if none).  Valid until the next call on ctx.
 * mr_last_error(NULL) describes the last failed mr_create. */
MR_API const char *mr_last_error(mr_ctx *ctx);

/* ---- problem set-up ("continuous energy total cross section data ... 3-D
 *      Cartesian mesh geometry"; geometry and tally share the mesh) ------------ */

/* Rectilinear mesh given by its plane positions: xe[nx+1], ye[ny+1], ze[nz+1], host, strictly
 * increasing, finite.  nx*ny*nz must be < 2^31 and each of nx, ny, nz <= 32767.  Allocates and zeroes the fp64 tally; drops
 * any material map loaded before.  Errors: INVALID_ARG, UNSUPPORTED, OOM, CUDA. */
MR_API int mr_load_mesh(mr_ctx *ctx, int nx, int ny, int nz, const double *xe, const double *ye, const double *ze);

/* R-Z (2-D cylindrical) tally mesh: nr radial shells re[0] = 0 < ... < re[nr]
 * about the z axis and nz axial slabs ze[0..nz]; cell (ir, iz) = { re[ir] <= sqrt(x^2+y^2) < re[ir+1], ze[iz] <= z <
 * ze[iz+1] }, linear index c = ir + nr*iz (ncell = nr*nz).  Rays stay 3-D records; everything else (materials,
 * tables, mr_cast_rays, mr_trace_rays, moments, the producer ring) works as on a Cartesian mesh, with the walk of
 * radial crossings from the quadratic (ox+t dx)^2 + (oy+t dy)^2 = r_p^2, ties radial before
 * axial; a ray is rejected if x^2+y^2 >= re[nr]^2 or z is outside [ze[0], ze[nz]).  mr_cast_next_event works too
 * (steps NZ1-NZ6 of DESIGN.md section 10.7: the same radial / axial crossings with the unnormalised direction towards the
 * detector).  Replaces any mesh loaded before.  Errors: INVALID_ARG (re[0] != 0, not increasing), UNSUPPORTED, OOM, CUDA. */
MR_API int mr_load_mesh_rz(mr_ctx *ctx, int nr, int nz, const double *re, const double *ze);

/* 1-D spherical tally mesh ("1-D spherical meshes"): nr shells re[0] = 0 < ... < re[nr] about the origin,
 * cell c = ir = the shell that holds sqrt(x^2+y^2+z^2) (ncell = nr).  The walk is the radial part of the R-Z walk with
 * rho0^2 = |o|^2, a = |d|^2, b = o.d and no axial crossings; a ray is rejected if |o|^2 >= re[nr]^2.  Same
 * restrictions as mr_load_mesh_rz.  Errors: INVALID_ARG, UNSUPPORTED, OOM, CUDA. */
MR_API int mr_load_mesh_sphere(mr_ctx *ctx, int nr, const double *re);

/* Materials and per-cell composition.  density[M] g/cc (finite, >= 0); K slots per cell;
 * cell_mat[ncell*K] material index per slot, -1 = empty slot; cell_frac[ncell*K] volume
 * fractions (finite, >= 0; ignored for empty slots).  Slot k of cell c is element c*K+k.
 * The library stores r = frac*density (rounded once to fp32 in MIXED mode) and the total
 * cross section of cell c at energy E is Sigma_t = sum_k r[c,k] * sigma_{mat[c,k]}(E), summed
 * in slot order (reading Q3).  Requires mr_load_mesh.  Drops loaded tables when M
 * changes.  All host arrays.  Errors: INVALID_ARG, STATE, UNSUPPORTED (M > MR_MAX_MATERIALS,
 * K > MR_MAX_SLOTS), OOM, CUDA. */
MR_API int mr_load_materials(mr_ctx *ctx, int M, const double *density, int K, const int32_t *cell_mat,
                      const double *cell_frac);

/* Tabulated total cross section of material `material`: energy[n] MeV strictly increasing and
 * > 0, sigma_t[n] cm^2/g finite and >= 0, host arrays, n >= 1.  sigma(E) is the lin-lin
 * interpolant, clamped to the end values outside the grid (reading Q5).
 * In MIXED mode the values are stored as fp32 (pass fp32-representable values to keep the
 * bracket identical to a double evaluation).  Requires mr_load_materials.
 * Errors: INVALID_ARG, STATE, OOM, CUDA. */
MR_API int mr_load_xs(mr_ctx *ctx, int material, int64_t n, const double *energy, const double *sigma_t);

/* Multi-nuclide materials ("first calculating all cross-sections"): instead of a
 * table of its own a material may be a mixture of nuclides, each with its own energy grid:
 *     sigma_m(E) = sum_j weights[j] * sigma_{nuclides[j]}(E)        (added in list order)
 * mr_load_nuclide_xs loads nuclide `nuclide`'s table (0 <= nuclide < MR_MAX_NUCLIDES; same rules as mr_load_xs; may be
 * called any time after mr_create); mr_define_material makes material `material` the mixture of nnuc (1..MR_MAX_MIX)
 * nuclides with the given weights (finite, >= 0; e.g. mass fractions, so that sigma stays in cm^2/g; stored as fp32 in
 * MIXED mode) and drops the material's own table, if any; a later mr_load_xs for that material drops the mixture.
 * mr_cast_rays needs the table of every nuclide a mixture names.  Errors: INVALID_ARG, STATE, OOM, CUDA. */
MR_API int mr_load_nuclide_xs(mr_ctx *ctx, int nuclide, int64_t n, const double *energy, const double *sigma);
MR_API int mr_define_material(mr_ctx *ctx, int material, int nnuc, const int32_t *nuclides, const double *weights);

/* ---- the hot path ------------------------------------------------------------------------ */

/* Casts a batch of n rays and ADDS their scores to the resident tally (PAPER.md:77-85,
 * Eq. (4)).  `rays` is an array of n records {x,y,z,u,v,w,E,W}: 8 floats in
 * MIXED mode, 8 doubles in DOUBLE mode; where = MR_WHERE_HOST or MR_WHERE_DEVICE (device
 * buffers must be 16-byte aligned).  W is the already divided weight W/N of Eq. (4).
 * For every accepted ray, with tau = 0 at the origin, for each crossed cell i in order:
 *     x = Sigma_i * l_i;   score = W * exp(-tau) * (x > 0 ? (1 - exp(-x)) / Sigma_i : l_i);
 *     tally[i] += score;   tau += x
 * until the ray leaves the mesh (no cut-off, no reflection: readings Q7, F5).  A ray is
 * REJECTED (counted, no contribution) if any field is not finite, E <= 0, no axis has a
 * finite 1/d_a (the zero vector, or components so small that every reciprocal overflows: an
 * axis whose 1/d_a is not finite never steps, reading Q10, and a ray that steps on no axis
 * never leaves the mesh), or the origin is outside the half-open box [lo, hi) on any axis.
 * Asynchronous: returns once the batch is staged (a host buffer has been copied out of, or,
 * if it is page-locked, DMA'd out of) and the work is queued.  n = 0 is a no-op.
 * Requires mesh, materials and all M tables.  Errors: INVALID_ARG, STATE, OOM, CUDA. */
MR_API int mr_cast_rays(mr_ctx *ctx, int64_t n, const void *rays, int where);

/* mr_cast_rays for a caller that must not allocate device memory while it runs.
 *
 * Who that is: a transport code that hands the whole GPU to its own memory pool at start-up, so that nothing is left for
 * a library to allocate from; a host loop that cannot afford the device-wide wait a cudaMalloc / cudaFree implies (it
 * breaks the CPU/GPU overlap of PAPER.md:79-83); a job with a fixed memory budget per process.  mr_cast_rays does
 * allocate on their hot path: its ray-ordering pre-pass keeps a key and a sorted position per ray plus a histogram in
 * scratch memory that is allocated on the first batch and re-allocated whenever a batch is larger than any before.
 *
 * This call does the same work -- same ordering keys, same cast kernels, same tally, same counters -- but its pre-pass
 * works in a fixed array inside the library image, so it calls no cudaMalloc, no cudaFree, not the context's
 * mr_allocator, and no library routine that allocates.  The price is a limit and a reservation: at most
 * MR_STATIC_MAX_RAYS (262 144) rays per call -- more is refused with MR_ERR_INVALID_ARG and a message, split the batch --
 * and 2.1 MB of device memory on EVERY GPU the process uses, held from the moment the library is loaded until the process
 * exits, whether or not this call is ever made.
 *
 * `d_rays`: n ray records in DEVICE memory (layout as mr_cast_rays, 16-byte aligned); the caller owns them and must
 * keep them alive and unchanged until the queued work has run.  The tally is the context's, as for mr_cast_rays;
 * the two calls can be mixed freely on one context.  Asynchronous; n = 0 is a no-op.
 *
 * Before the first call: all allocation belongs to set-up.  Load mesh, materials and tables, then make ONE ordinary
 * mr_cast_rays call (a single ray is enough): it creates the small table-descriptor buffers.  Until that has happened
 * this call returns MR_ERR_STATE.  Tables re-loaded later are picked up without allocating.
 * First call on each device: looks up the device address of the fixed array (once per device, with the context's device
 * current).  Make that first call outside any stream capture.
 *
 * Sharing: there is one array per GPU, not per context or stream, and every call leaves its keys and positions in it (the
 * part that has to start at zero, the histogram, is cleared by each call on the context's stream).  Calls whose GPU work
 * can run at the same time -- two contexts on one GPU, or one context switched to another stream by mr_set_stream while
 * an earlier call is still in flight -- race on it and scramble each other's ray order.  Serialise them: one context
 * per GPU on one stream, or an event / mr_sync between calls from different contexts.
 *
 * Not available for R-Z / spherical meshes, nor when the deferred two-phase tally is active (MR_INFO_DEFERRED = 1; its pair
 * pool is sized per batch -- set MR_OPT_DEFERRED_TALLY to 0): MR_ERR_UNSUPPORTED.  Not while a producer ring is open:
 * MR_ERR_STATE.  mr_stats.last_kernel_ms reads 0 after this call (the per-kernel event list is not grown here);
 * last_cast_ms covers pre-pass + cast.  Errors: INVALID_ARG, STATE, UNSUPPORTED, CUDA. */
MR_API int mr_cast_rays_static(mr_ctx *ctx, int64_t n, const void *d_rays);

/* Synchronises and copies the ncell raw fp64 sums to the host array `out` ("the
 * tally remained on the GPU until the termination of the simulation").  A consistent
 * snapshot: all work queued before the call is included.  Errors: INVALID_ARG, STATE, CUDA. */
MR_API int mr_read_tally(mr_ctx *ctx, double *out);

/* The same snapshot without waiting for it: a device-side copy of the tally is taken in stream order (it holds exactly the
 * work queued before this call) and copied to `out` on a stream of its own, so that the transfer overlaps the casts
 * queued AFTER the call -- a host loop that casts batch after batch and wants every batch's running tally on the host
 * pays for the read-back once, at the end, instead of once per batch (the paper's own flow reads the tally only at the
 * end).  `out` (ncell doubles; page-locked memory if the copy is to be asynchronous) is valid after the next
 * mr_sync or mr_read_tally; a second mr_read_tally_async waits, on the device, for the first to have left the snapshot
 * buffer.  Allocates ncell doubles of device memory on first use.  Errors: INVALID_ARG, STATE, OOM, CUDA. */
MR_API int mr_read_tally_async(mr_ctx *ctx, double *out);

/* Zeroes the tally and the ray/segment counters (queued on the stream). */
MR_API int mr_clear_tally(mr_ctx *ctx);

/* Blocks until all queued work of the context has finished, pending mr_read_tally_async transfers included. */
MR_API int mr_sync(mr_ctx *ctx);

/* Synchronises and fills *out. */
MR_API int mr_get_stats(mr_ctx *ctx, mr_stats *out);

/* Borrowed device pointer to the ncell fp64 tally (e.g. for a caller-side NCCL all-reduce
 * across replicas).  Valid until the next mr_load_mesh / mr_destroy.  The call brings the array up to date
 * (work queued on the context's stream) and, from then on until the next mr_load_mesh, every cast adds
 * straight into it: the score accumulators of MR_OPT_FUSED_TALLY and MR_OPT_TILED_TALLY, which live outside
 * this array, are no longer used, so a view the caller keeps goes on following the tally in stream order. */
MR_API int mr_tally_device_ptr(mr_ctx *ctx, double **out);

/* ---- per-batch moments (Eq. (5) FOM = 1/(sigma^2 T), "sigma the
 *      standard deviation of the tally mean") -------------------------------------------------- */

/* Closes a batch: with x_b[c] = what was added to tally[c] since the previous mr_end_batch (or since
 * creation / mr_clear_tally), accumulates sumsq[c] += x_b[c]^2 on the device and counts the batch.  The
 * tally itself stays the running total (sum_b x_b), so mr_read_tally is unchanged.  Queued on the stream.
 * The first call allocates two more ncell-double arrays.  Errors: STATE (no mesh), OOM, CUDA. */
MR_API int mr_end_batch(mr_ctx *ctx);

/* Synchronises and returns the moments over the CLOSED batches: sum[c] = sum_b x_b[c] (the tally as of the
 * last mr_end_batch), sumsq[c] = sum_b x_b[c]^2, *nbatch = B.  Host arrays of ncell doubles; any of the
 * three may be NULL.  Before the first mr_end_batch: zeros and B = 0.  Errors: STATE, CUDA. */
MR_API int mr_read_moments(mr_ctx *ctx, double *sum, double *sumsq, int64_t *nbatch);

/* Synchronises, evaluates on the device and returns per cell the batch mean  mean = sum/B  and the standard
 * deviation OF THE MEAN  sigma = sqrt(max((sumsq/B - mean^2)/(B-1), 0))  (+inf when B = 1), the sigma of
 * Eq. (5).  Host arrays of ncell doubles, either may be NULL.  Errors: STATE (no closed batch), OOM, CUDA. */
MR_API int mr_read_mean_sigma(mr_ctx *ctx, double *mean, double *sigma, int64_t *nbatch);

/* ---- next-event (point-detector) estimator ("requires a ray-cast
 *      from each source and collision event to the estimator location") ------------------------ */

/* Detector points xyz[ndet*3] (host, finite; inside or outside the mesh).  Allocates and zeroes the ndet
 * resident fp64 detector sums and the next-event counters; replaces any earlier set.  1 <= ndet <= 65535.
 * Errors: INVALID_ARG, UNSUPPORTED, OOM, CUDA. */
MR_API int mr_load_detectors(mr_ctx *ctx, int ndet, const double *xyz);

/* For every event (the same records as mr_cast_rays; only x,y,z,E,W are used, the direction fields are
 * ignored) and every detector d: with dvec = det_d - origin (fp64), R^2 = |dvec|^2, the cells between the
 * origin and the detector are walked exactly as in mr_cast_rays but with the unnormalised direction dvec,
 * so the crossing parameter t = 1 IS the detector; the segment whose pending crossing has t >= 1 ends at
 * the detector and is the last; leaving the mesh ends the walk too (outside the mesh is void);
 *     tau = sum_i Sigma_i * (l_i * R);     det_sum[d] += W * exp(-tau) / R^2
 * W must already carry the angular density p(Omega -> detector) of the event (reading N-Q1).
 * A pair is REJECTED (counted, no contribution) if x,y,z,E or W is not finite, E <= 0, the origin is outside
 * the half-open box, or R^2 is 0 or not finite.  Asynchronous like mr_cast_rays.  n = 0 is a no-op.
 * On an R-Z or spherical mesh the cells between event and detector are those of the mesh's own walk (radial crossings
 * from the quadratic in t, ties radial before axial), with the same unnormalised direction and the same end at t = 1; the
 * origin test is the mesh's (x^2+y^2 < re[nr]^2, z inside; |o|^2 < re[nr]^2 on a spherical mesh).
 * Requires mesh, materials, all tables and detectors.  Errors: INVALID_ARG, STATE, OOM, CUDA. */
MR_API int mr_cast_next_event(mr_ctx *ctx, int64_t n, const void *rays, int where);

/* Synchronises and copies the ndet detector sums to the host array `out`. */
MR_API int mr_read_detectors(mr_ctx *ctx, double *out);

/* Zeroes the detector sums and the next-event counters (queued on the stream). */
MR_API int mr_clear_detectors(mr_ctx *ctx);

/* Test entry: the same walk for ONE detector `det`, nothing is added to the detector sums or counters.  Per event r (host
 * outputs, any may be NULL): nseg[r] cells crossed (0 if rejected), hash[r] FNV-1a 64 of the cell sequence
 * (0 if rejected), tau[r], score[r].  Synchronous. */
MR_API int mr_trace_next_event(mr_ctx *ctx, int64_t n, const void *rays, int where, int det, uint32_t *nseg,
                               uint64_t *hash, double *tau, double *score);

/* ---- producer ring (Fig. 4: "rays were stored in a buffer and
 *      transferred to the GPU when the buffer became full ... the CPU cleared the buffer and resumed";
 *      one buffer per node shared by the ranks that feed one GPU) ------------------- */

typedef struct {
    int64_t rays_pushed;      /* rays accepted by mr_ring_push since mr_ring_open */
    int64_t slots_shipped;    /* buffers handed to the GPU (full ones and flushed partial ones) */
    double producer_wait_ms;  /* total time producers spent blocked because every slot was in flight */
    int64_t casts;            /* cast launches (each with its ordering pre-pass) the shipped buffers were merged into */
    double reserved[2];
} mr_ring_stats;

/* Opens a ring of `slots` (2..16) page-locked host buffers of `rays_per_slot` rays each (>= 1024), with as many
 * device buffers behind them.  Producers append rays with mr_ring_push; a buffer that becomes full is shipped:
 * H2D copy on the copy stream, then the ordering pre-pass and the cast kernel on the context's stream, without
 * blocking the producer -- which goes on filling the next buffer while the GPU works (Fig. 4).  A producer
 * blocks only when every buffer is still being copied out.  While an earlier cast of the ring is still running, a
 * shipped buffer is copied at once but its cast is held back and merged with the buffers that follow it into ONE
 * launch (MR_OPT_RING_MERGE; the device buffers are consecutive pieces of one allocation): the GPU is busy anyway,
 * and one cast of k buffers is cheaper than k casts.  mr_ring_flush queues whatever is held back.  Requires mesh, materials and all tables.
 * Errors: INVALID_ARG, STATE (ring already open, set-up incomplete), OOM, CUDA. */
MR_API int mr_ring_open(mr_ctx *ctx, int slots, int64_t rays_per_slot);

/* Appends n rays (HOST array of the context's record type) to the ring.  THREAD-SAFE: any number of host
 * threads may push concurrently (space is reserved under a lock, the copy into the page-locked buffer runs
 * outside it); this is the only entry point, with mr_ring_flush, that may be called while other threads are
 * inside the same context, and no other mr_* call may run at the same time.  The rays are consumed when the
 * call returns.  n may exceed a buffer.  Errors: INVALID_ARG, STATE (ring not open), CUDA. */
MR_API int mr_ring_push(mr_ctx *ctx, int64_t n, const void *rays);

/* Ships the partly filled buffer, if any.  After mr_ring_flush (and once every producer has returned from its
 * last push) all pushed rays are queued on the context's stream: mr_read_tally then includes them. */
MR_API int mr_ring_flush(mr_ctx *ctx);

/* Flushes, waits for the copies and frees the ring. */
MR_API int mr_ring_close(mr_ctx *ctx);

MR_API int mr_ring_get_stats(mr_ctx *ctx, mr_ring_stats *out);

/* Measurement aid for Fig. 4's overlap (the CPU goes on filling the next buffer while the GPU works on
 * the last one): `producers` (1..256) host threads created INSIDE the library push the n rays of the HOST array `rays`
 * through mr_ring_push in pieces of rays_per_push rays (thread k owns the k-th contiguous share), then mr_ring_flush is
 * called; *wall_ms (may be NULL) = wall-clock time from the first push to the return of the flush (the GPU work it queued
 * may still be running: mr_read_tally waits for it).  dry_run != 0: the threads copy the same pieces into private
 * scratch buffers instead -- no ring, no GPU: what the producers alone cost.  Requires an open ring unless dry_run.
 * Errors: INVALID_ARG, STATE (ring not open), and those of mr_ring_push / mr_ring_flush. */
MR_API int mr_ring_bench_producers(mr_ctx *ctx, int64_t n, const void *rays, int producers, int64_t rays_per_push, int dry_run,
                                   double *wall_ms);

/* ---- test / diagnostic entry point ------------------------------------------------------- */

/* The same walk as mr_cast_rays with no tally update.  Per ray r (host outputs, any may be
 * NULL): nseg[r] = number of segments (0 if rejected); hash[r] = FNV-1a 64 over the
 * little-endian bytes of the 32-bit cell indices in crossing order (0 if rejected);
 * if cap > 0: cells[r*cap + j], lens[r*cap + j] for the first min(nseg, cap) segments
 * (untouched beyond).  Needs only the mesh.  Synchronous.  Errors as mr_cast_rays. */
MR_API int mr_trace_rays(mr_ctx *ctx, int64_t n, const void *rays, int where, uint32_t *nseg, uint64_t *hash,
                  int32_t *cells, double *lens, int64_t cap);

/* ---- tuning knobs (never change results beyond fp64 summation order) ---------------------- */
enum {
    MR_OPT_BLOCK_THREADS = 1, /* threads per CTA of the cast kernel (multiple of 32, <= 256) */
    MR_OPT_SORT_RAYS = 2,     /* 0: cast in buffer order; 1: bin rays by start slab and length first */
    MR_OPT_STAGE_RAYS = 3,    /* base chunk size (rays) for host batches: chunks grow from a quarter of it to twice it; the H2D copy of
                                 chunk i+1 overlaps the cast of chunk i, and consecutive casts run on two internal lanes */
    MR_OPT_COPY_THREADS = 4,  /* host threads that copy a PAGEABLE batch into the pinned ring (a pinned batch is DMA'd directly) */
    MR_OPT_PAIR_RECORDS = 5,  /* 1: 16-byte cell records (K = 2, 3, MIXED) are fetched as 32-byte pairs kept in registers; 0: one by one */
    MR_OPT_ORDER_MODE = 6,    /* key of the MR_OPT_SORT_RAYS pre-pass: 1 = (start z-slab, length): CTAs resident together work in the
                                 same slabs (L2 reuse); 2 = longest rays first: no tail; 0 = auto: 2 when tally + cell records fit
                                 in half the L2, else 1 */
    MR_OPT_FUSED_TALLY = 7,   /* read by mr_load_materials.  K = 4 records (MIXED) have 8 spare bytes: 1 = the cast kernel accumulates
                                 each cell's score THERE (the load and the atomic of a segment then share one DRAM sector) and the sums
                                 are moved into the contiguous tally whenever it is looked at (mr_read_tally, mr_tally_device_ptr,
                                 mr_end_batch, mr_clear_tally); 0 = never; 2 (default) = when ncell * 40 bytes exceed twice the L2 */
    MR_OPT_TILED_INDEX = 8,   /* 1 (default): when a mesh (K <= 3, MIXED, Cartesian) holds at most 1024 DISTINCT cell records,
                                 mr_load_materials also builds a dictionary of them and a 2-byte index per cell in 32-byte tiles of
                                 4 x 4 (x, y) cells, and mr_cast_rays walks those (a step inside a tile needs no load); 0: never.
                                 Setting 0 after the load makes the cast use the plain records again */
    MR_OPT_COARSE_RECORDS = 10, /* read by mr_load_materials and mr_cast_rays.  1 (default): when every aligned block of 2^s cells per axis
                                 (largest s in 1..5; MIXED, K <= 4, Cartesian, no dictionary path) holds ONE composition -- a material map
                                 coarser than the tally mesh -- mr_load_materials also stores one record per BLOCK and mr_cast_rays reads
                                 those: the table stays in L2 where per-cell records of a mesh far larger than L2 cost a DRAM line per
                                 segment, and a step inside a block needs no load.  0: never (after the load: use the per-cell records) */
    MR_OPT_DEFERRED_TALLY = 11, /* the two-phase tally for meshes far larger than L2 (MIXED, Cartesian; coarse-record or K = 4 record path):
                                 phase A walks and scores but appends (cell, score) pairs to the bin of the cell's tally REGION (a range
                                 of the linear cell index worth at most L2/8 of tally), phase B adds the pairs bin after bin, while the
                                 region is in L2.  tally[c] receives the same scores in another order.  0 = never, 1 = whenever the
                                 path allows, 2 (default) = coarse-record path on a mesh whose tally exceeds twice the L2 */
    MR_OPT_DEFER_POOL_ENTRIES = 12, /* size of the deferred tally's pool in (cell, score) pairs (12 bytes each); 0 (default) = sized from the batch
                                 (rays x (nx+ny+nz)/3, at most 24 GB; batches that need more are cast in pieces) and grown when a cast ran
                                 out.  A pool that is too small is never an error: the pairs that do not fit are added straight to the tally */
    MR_OPT_DEFER_REGION_SHIFT = 13, /* s: the deferred tally's regions are 2^s cells of the linear cell index (at most 64 regions: s is raised
                                 until they cover the mesh); 0 (default) = the largest s with 8 * 2^s bytes <= L2/8 */
    MR_OPT_COOP_FLUSH = 14,   /* 1: the cast kernel stages every lane's (cell, score) pairs for 8 steps in shared memory and the warp then
                                 adds them TRANSPOSED, one instruction carrying 8 consecutive segments of each of 4 rays (consecutive
                                 cells of a ray often share a 32-byte tally sector; cells of unrelated rays never do).  MIXED mode:
                                 dictionary / K = 1 / K = 3 pairs / dense-8 record paths; DOUBLE mode: the K <= 3 record path;
                                 elsewhere ignored.  0: one atomic per
                                 segment straight from the walking lane.  2 (default) = auto: on when tally + cell records fit in
                                 half the L2 (it wins there: contended, resident tallies) and on the K = 3 record-pair path and the
                                 DOUBLE-mode K <= 3 path at any size, off elsewhere.  3 = the same idea with pairs instead of windows of 8: every lane walks two steps
                                 and swaps one (cell, score) pair with its neighbour lane by shuffles (no shared memory; measured
                                 no better than 1 anywhere) */
    MR_OPT_RZ_BLOCK_THREADS = 15, /* threads per CTA of the R-Z / spherical cast kernel (multiple of 32, <= 256; default 256: every CTA stages
                                 the mesh's radii and planes in shared memory) */
    MR_OPT_TILED_TALLY = 16,  /* 1: on the dictionary path (MR_OPT_TILED_INDEX) the cast kernel keeps the walk in tile coordinates
                                 and adds the scores into TILE-ORDERED accumulators (one double per tile entry: consecutive cells of a ray
                                 are neighbours in memory whichever of x and y the ray steps in), which are moved into the linear tally
                                 whenever it is looked at (mr_read_tally, mr_tally_device_ptr, mr_end_batch, mr_clear_tally); with
                                 MR_OPT_COOP_FLUSH the transposed adds then share 128-byte lines (L2 requests per segment 1.0 -> 0.45).
                                 0 (default): the kernel adds straight into the linear tally -- measured faster on every config
                                 (the kernel is bound by instruction issue once the requests are gone) */
    MR_OPT_WHOLE_BATCH = 18,  /* page-locked HOST batches of mr_cast_rays: 0 = always the chunked pipeline of MR_OPT_STAGE_RAYS (the first kernel
                                 starts after a short copy: lowest latency of a call on an idle GPU); 1 = always one DMA of the whole batch
                                 into one of two device buffers and ONE cast behind it; 2 (default) = auto: whole-batch when the context's
                                 stream is still busy with earlier work when the call is made (a caller casting batch after batch without
                                 waiting: the copy then hides behind the previous cast, and one launch is 20 % cheaper than its chunks),
                                 chunked otherwise.  Batches above 2 GB are always chunked */
    MR_OPT_RING_MERGE = 19,   /* producer ring: 0 = every shipped buffer gets its own ordering pre-pass and cast; 1 (default) = auto: a buffer
                                 shipped while an earlier cast of the ring is still running waits, and consecutive waiting buffers are cast
                                 in one launch by the next ship that finds the GPU free, by a ship that wraps around the ring, or by
                                 mr_ring_flush; 2 = always wait (one cast per ring revolution or flush).  Set before mr_ring_open */
    /* 17 was MR_OPT_PERSISTENT_LANES (a cast kernel whose lanes refilled from a counter): measured slower on every config
        and removed in round 3 */
    MR_OPT_AGGREGATE_FIRST = 9 /* n >= 0: the tally atomics of the first n segments of every ray are warp-aggregated (lanes that score
                                 into the same cell are found with match.any and one of them adds the sum): for batches born in a
                                 region of a few cells, where same-address atomics serialise in L2.  Default 2; 0 = off */
};
/* Read-only facts about the resident problem, through mr_get_option (mr_set_option refuses them). */
enum {
    MR_INFO_RECORD_PATH = 100,     /* which cell-record path (S4) mr_cast_rays takes now: one of MR_PATH_* */
    MR_INFO_DISTINCT_RECORDS = 101,/* size of the dictionary of distinct cell records (0: none was built) */
    MR_INFO_COARSE_SHIFT = 102,    /* s of MR_OPT_COARSE_RECORDS (blocks of 2^s cells per axis; 0: none) */
    MR_INFO_DEFERRED = 103,        /* 1 if mr_cast_rays uses the deferred tally now (MR_OPT_DEFERRED_TALLY) */
    MR_INFO_DEFER_DIRECT_PAIRS = 104 /* (cell, score) pairs the deferred tally had to add directly because its pool was full */
};
enum {
    MR_PATH_NONE = 0,          /* no materials loaded */
    MR_PATH_K1 = 1,            /* MIXED, 8-byte records {r, id} */
    MR_PATH_K2 = 2,            /* MIXED, 16-byte records, one load per cell */
    MR_PATH_K3 = 3,
    MR_PATH_K4 = 4,            /* MIXED, 32-byte records */
    MR_PATH_K2_PAIRS = 5,      /* MIXED, 16-byte records fetched as 32-byte x-neighbour pairs (MR_OPT_PAIR_RECORDS) */
    MR_PATH_K3_PAIRS = 6,
    MR_PATH_K4_FUSED = 7,      /* MIXED, 32-byte records that also hold the cell's score accumulator (MR_OPT_FUSED_TALLY) */
    MR_PATH_DENSE8 = 8,        /* MIXED, K = M = 8, ids implicit */
    MR_PATH_GENERIC = 9,       /* MIXED, coefficient + id arrays */
    MR_PATH_TILED4 = 10,       /* MIXED, dictionary + tiled index, 4-bit / 8-bit / 16-bit indices (MR_OPT_TILED_INDEX) */
    MR_PATH_TILED8 = 11,
    MR_PATH_TILED16 = 12,
    MR_PATH_COARSE = 13,       /* MIXED, one record per block of cells (MR_OPT_COARSE_RECORDS) */
    MR_PATH_DOUBLE_K3 = 14,    /* DOUBLE, K <= 3, 32-byte records */
    MR_PATH_DOUBLE_GENERIC = 15,
    MR_PATH_RZ = 16            /* R-Z / spherical mesh kernel (per-cell records of the layouts above) */
};
MR_API int mr_set_option(mr_ctx *ctx, int option, int64_t value);
MR_API int mr_get_option(mr_ctx *ctx, int option, int64_t *value);

/* ---- measurement aid ------------------------------------------------------------------------ */

/* The L2 fp64-atomic ceiling the cast kernel is measured against ("L2 atomic throughput against a
 * measured micro-benchmark").  Issues the cast kernel's per-segment memory pattern and nothing else: every lane adds into
 * a pseudo-random cell of a scratch array of `ncell` doubles (red.global.add.f64), optionally after loading `gather_bytes`
 * (0, 16 or 32) from a scratch record array at the same cell; lanes in groups of `group` (a power of two <= 32) take
 * consecutive cells (group = 4: one 32-byte sector).  ceil(lane_ops / 8192) * 8192 lane operations per launch, two warm-up
 * launches, then `reps` timed ones on the legacy default stream of `device`: *best_ms and *mean_ms (may be NULL) per launch.
 * Needs no context; allocates and frees its own scratch.  Errors: INVALID_ARG, CUDA, OOM. */
MR_API int mr_microbench_red(int device, int64_t ncell, int group, int gather_bytes, int64_t lane_ops, int reps,
                             double *best_ms, double *mean_ms);

#ifdef __cplusplus
}
#endif
#endif /* MONTERAY_H */
