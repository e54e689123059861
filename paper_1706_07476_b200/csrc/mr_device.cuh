// mr_device.cuh -- device code of the VRC ray-cast hot path (sm_100a).
//
// Steps S1..S6 of DESIGN.md §1 ("first calculating all cross-sections, then ray
// casting the particle, and finally calculating the VRC estimator", Eq. (4)).
// Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

namespace mr {

// ------------------------------------------------------------------------------------------------
// Kernel parameter blocks (plain data, passed by value)
// ------------------------------------------------------------------------------------------------
struct XsDesc {            // one material's table (device pointers)
    const void *E;         // float[n] (mixed) or double[n]
    const void *S;
    int n;
    int grid;              // materials whose energy grids are bitwise identical share a grid id (and E, first)
    // bucket index of the grid (the paper's hash-based lookup): bucket(E) = (bits((float)E) >> sh) - b0
    // is non-decreasing in E; first[b] = number of grid points whose bucket is < b, for b = 0..nb
    const uint32_t *first;
    uint32_t b0;
    int sh;
};

enum CellLayout : int {
    LAYOUT_K1 = 1,         // 8 B  {float r; u32 id}
    LAYOUT_K2 = 2,         // 16 B {float r0,r1; u32 ids; u32 pad}
    LAYOUT_K3 = 3,         // 16 B {float r0,r1,r2; u32 ids}
    LAYOUT_K4 = 4,         // 32 B {float r0..r3; u32 ids; u32 pad[3]}
    LAYOUT_D8 = 8,         // 32 B {float r[8]}  dense: slot k holds material k
    LAYOUT_DK3 = 23,       // DOUBLE mode, K <= 3: 32 B {double r0,r1,r2; u32 ids; u32 pad}, one LDG.E.256 per cell
    LAYOUT_T3 = 15,        // kernel-side only: dictionary of distinct K <= 3 records + tiled 2-byte index per cell
    LAYOUT_K4F = 14,       // kernel-side only: LAYOUT_K4 record whose 8 spare bytes (offset 24) hold the cell's score accumulator
    LAYOUT_K2P = 12,       // kernel-side only: LAYOUT_K2 / LAYOUT_K3 records fetched as 32-byte pairs
    LAYOUT_K3P = 13,
    LAYOUT_C4 = 16,        // kernel-side only: block-constant compositions -- LAYOUT_K4 records on a coarse grid of 2^s-cell blocks
    LAYOUT_GENERIC = 100   // coef[ncell*K] (float or double) + ids[ncell*K] (u8, 0xff = empty)
};

struct MeshDev {
    int nx, ny, nz;
    int nedges;            // nx+1 + ny+1 + nz+1
    const double *edges;   // x planes | y planes | z planes, concatenated
    // "arithmetic" axes: mr_load_mesh verified edges_a[p] == fma((double)p, h[a], e0[a]) bit for bit for
    // every plane, so the walker may recompute a plane position instead of looking it up
    double e0[3], h[3];
};

// where the walker finds plane positions
enum EdgeMode : int { EDGES_GLOBAL = 0, EDGES_SHARED = 1, EDGES_ARITH = 2 };

struct CastParams {
    MeshDev mesh;
    const void *recs;      // packed records (LAYOUT_K*, LAYOUT_D8) or coefficient array (generic)
    const uint8_t *ids;    // generic layout only
    const uint4 *dict;     // LAYOUT_T3: the distinct records (K = 3 encoding), ndict of them
    const uint4 *tiles;    // LAYOUT_T3: 32-byte tiles of 4 x 4 (x, y) 2-byte dictionary indices, ntx * nty * nz of them
    int ndict, ntx, nty;
    const void *crecs;     // LAYOUT_C4: one LAYOUT_K4 record per block of 2^cshift cells per axis, cnx * cny * cnz of them
    int cshift, cnx, cny;
    int K, M;
    const XsDesc *xs;      // [M + N]: materials (n = 0: a nuclide mixture), then nuclides
    int N;                 // nuclide descriptors (0: every material has a table of its own)
    const int *mix_off;    // [M + 1] entries of material m: mix_off[m] .. mix_off[m+1]-1
    const int *mix_nuc;    // nuclide per entry
    const void *mix_w;     // weight per entry (Real)
    const void *rays;      // 8 floats (mixed) or 8 doubles per ray
    const uint32_t *perm;  // optional processing order (ray index per work item), may be null
    long long n;
    int agg_first;         // warp-aggregate the tally atomics of the first agg_first segments of every ray (0: never)
    double *tally;
    double *tally_t;       // dictionary path with tile-ordered accumulators (mr_tiled.cuh): acc[tile * cells_per_tile + entry]
    unsigned long long *counters;  // [0] accepted [1] rejected [2] segments
};

struct TraceParams {
    MeshDev mesh;
    const void *rays;
    long long n;
    uint32_t *nseg;        // may be null
    unsigned long long *hash;  // may be null
    int32_t *cells;        // may be null, [n*cap]
    double *lens;          // may be null, [n*cap]
    long long cap;
    int ray_is_double;
};

// ------------------------------------------------------------------------------------------------
// Small helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float4 ldg_f4(const void *p) { return __ldg(reinterpret_cast<const float4 *>(p)); }
// Cell records are read once per segment by lanes that are 32 unrelated rays: a line brought into L1 is almost never hit
// again (L1 hit rate 4 %), so the record loads bypass L1 allocation (ld.global.nc.L1::no_allocate).  Measured on config 3:
// cast kernel 8.83 -> 8.41 ms.
__device__ __forceinline__ uint4 ldg_u4(const void *p)
{
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ uint2 ldg_u2(const void *p)
{
    uint2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ double2 ldg_d2(const void *p) { return __ldg(reinterpret_cast<const double2 *>(p)); }

// 32-byte read-only load (LDG.E.256 on sm_100a); p must be 32-byte aligned
__device__ __forceinline__ void ldg_256(const void *p, uint4 &lo, uint4 &hi)
{
    asm volatile("ld.global.nc.L1::no_allocate.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(lo.x), "=r"(lo.y), "=r"(lo.z), "=r"(lo.w), "=r"(hi.x), "=r"(hi.y), "=r"(hi.z), "=r"(hi.w)
                 : "l"(p));
}

// fp64 reduction into global memory without a return value (RED.E.ADD.F64 in SASS)
__device__ __forceinline__ void red_add_f64(double *addr, double v)
{
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(addr), "d"(v) : "memory");
}

// Ray record {x,y,z,u,v,w,E,W} -> doubles (exact promotion in mixed mode).  Returns the O1
// validation verdict except for the box test (done by the walker once the mesh is known).
template <typename Real>
struct Ray {
    double o[3], d[3];
    Real E;
    double W;
    bool finite;
};

__device__ __forceinline__ Ray<float> load_ray_f32(const void *rays, long long r)
{
    const float4 *p = reinterpret_cast<const float4 *>(rays) + 2 * r;
    float4 a = __ldg(p), b = __ldg(p + 1);
    Ray<float> R;
    R.o[0] = a.x; R.o[1] = a.y; R.o[2] = a.z;
    R.d[0] = a.w; R.d[1] = b.x; R.d[2] = b.y;
    R.E = b.z; R.W = b.w;
    R.finite = isfinite(a.x) && isfinite(a.y) && isfinite(a.z) && isfinite(a.w) && isfinite(b.x) &&
               isfinite(b.y) && isfinite(b.z) && isfinite(b.w);
    return R;
}

__device__ __forceinline__ Ray<double> load_ray_f64(const void *rays, long long r)
{
    const double2 *p = reinterpret_cast<const double2 *>(rays) + 4 * r;
    double2 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2), e = __ldg(p + 3);
    Ray<double> R;
    R.o[0] = a.x; R.o[1] = a.y; R.o[2] = b.x;
    R.d[0] = b.y; R.d[1] = c.x; R.d[2] = c.y;
    R.E = e.x; R.W = e.y;
    R.finite = isfinite(a.x) && isfinite(a.y) && isfinite(b.x) && isfinite(b.y) && isfinite(c.x) &&
               isfinite(c.y) && isfinite(e.x) && isfinite(e.y);
    return R;
}

template <typename Real> __device__ __forceinline__ Ray<Real> load_ray(const void *rays, long long r);
template <> __device__ __forceinline__ Ray<float> load_ray<float>(const void *rays, long long r) { return load_ray_f32(rays, r); }
template <> __device__ __forceinline__ Ray<double> load_ray<double>(const void *rays, long long r) { return load_ray_f64(rays, r); }

// ------------------------------------------------------------------------------------------------
// S1: sigma_m(E), lin-lin interpolation in a table, end values outside (Q5).
// The bracket k (E_k <= E < E_{k+1}) is the one a plain upper_bound gives (reading Q4); the bucket index
// only narrows the range the binary search starts from: every grid point in a lower bucket is < E and
// every point in a higher bucket is > E because bucket() is monotone.  Materials that share a grid share
// the bracket and the interpolation weight, so the search runs once per distinct grid.
// ------------------------------------------------------------------------------------------------
template <typename Real>
struct Bracket {
    int k;       // -1: E below the grid (or n == 1), -2: E at or above the last point, else the bracket
    Real t01;    // (E - E_k) / (E_{k+1} - E_k)
};

template <typename Real>
__device__ __forceinline__ Bracket<Real> find_bracket(const XsDesc &t, Real E)
{
    const Real *__restrict__ Eg = reinterpret_cast<const Real *>(t.E);
    const int n = t.n;
    Bracket<Real> b;
    b.t01 = (Real)0;
    if (n == 1 || E < __ldg(Eg)) { b.k = -1; return b; }
    if (E >= __ldg(Eg + n - 1)) { b.k = -2; return b; }
    const uint32_t bk = (__float_as_uint((float)E) >> t.sh) - t.b0;
    int lo = max((int)__ldg(t.first + bk), 1), hi = min((int)__ldg(t.first + bk + 1), n - 1);
    while (lo < hi) {        // invariant: Eg[lo-1] <= E < Eg[hi]
        const int mid = (lo + hi) >> 1;
        if (__ldg(Eg + mid) <= E) lo = mid + 1; else hi = mid;
    }
    b.k = lo - 1;            // Eg[k] <= E < Eg[k+1], 0 <= k <= n-2
    const Real e0 = __ldg(Eg + b.k), e1 = __ldg(Eg + b.k + 1);
    b.t01 = (E - e0) / (e1 - e0);
    return b;
}

template <typename Real>
__device__ __forceinline__ Real sigma_at(const XsDesc &t, const Bracket<Real> &b)
{
    const Real *__restrict__ Sg = reinterpret_cast<const Real *>(t.S);
    if (b.k == -1) return __ldg(Sg);
    if (b.k == -2) return __ldg(Sg + t.n - 1);
    const Real s0 = __ldg(Sg + b.k), s1 = __ldg(Sg + b.k + 1);
    return s0 + b.t01 * (s1 - s0);
}

// S1 for a whole ray ("first calculating all cross-sections"): sigma of every material into the
// thread's shared column sig[m * stride], m < M.  With nuclides (N > 0) the nuclide values go to columns
// M .. M+N-1 first and a mixture material is the weighted sum of its nuclides, added in list order.
template <typename Real>
__device__ __forceinline__ void sigma_all(const XsDesc *xs, int M, int N, const int *mix_off, const int *mix_nuc,
                                          const void *mix_w, Real E, Real *sig, int stride)
{
    Bracket<Real> br;
    int grid = -1;
    for (int q = M; q < M + N; ++q) {
        const XsDesc t = xs[q];
        if (t.n == 0) continue;                     // nuclide not loaded (and, checked on the host, not used)
        if (t.grid != grid) { br = find_bracket<Real>(t, E); grid = t.grid; }
        sig[q * stride] = sigma_at<Real>(t, br);
    }
    for (int m = 0; m < M; ++m) {
        const XsDesc t = xs[m];
        if (t.n > 0) {
            if (t.grid != grid) { br = find_bracket<Real>(t, E); grid = t.grid; }
            sig[m * stride] = sigma_at<Real>(t, br);
        } else {
            const Real *w = reinterpret_cast<const Real *>(mix_w);
            Real s = 0;
            for (int j = __ldg(mix_off + m); j < __ldg(mix_off + m + 1); ++j)
                s += __ldg(w + j) * sig[(M + __ldg(mix_nuc + j)) * stride];
            sig[m * stride] = s;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S2 + S3: the walker.  Crossing parameter of plane p on axis a is the pure function
//   t_a(p) = (edges_a[p] - o_a) * inv_a          (one subtract, then one multiply, both RN)
// and the trace is the 3-way merge of the three non-decreasing sequences, ties x < y < z
// (O3-O5).  __dsub_rn/__dmul_rn keep the compiler from contracting anything.
//
// State: the three pending crossing parameters, the current parameter, the cell index, and per
// axis one packed word (next plane | exit plane << 16) and the signed cell-index increment live in
// registers; the per-axis doubles (o_a, inv_a) sit in shared memory, [axis][thread], 16 B each, so a
// warp's LDS.128 is bank-conflict free whatever axis each lane picks.  The kernel is bound by
// per-request units (LSU wavefronts, the SM->L2 request port, L2 tag look-ups: DESIGN.md §4.3, §4.6), so shared-memory
// traffic per step is kept to that one LDS.128 (+ the sigma reads); when the mesh is arithmetic
// (EDGES_ARITH) the plane position is recomputed with one I2F + DFMA instead of a table read.
// ------------------------------------------------------------------------------------------------
struct __align__(16) AxisF { double o, iv; };

struct Walker {
    double t0, t1, t2;     // pending crossing parameter per axis (+inf: the axis never steps)
    double tcur;
    int c;                 // current cell
    int pl0, pl1, pl2;     // next plane (low 16 bits) | plane whose crossing leaves the mesh (high 16 bits)
    int dc0, dc1, dc2;     // signed cell-index increment of a step (sign = step direction; 0: never steps)
};

// number of entries of e[0..n) that are <= v
__device__ __forceinline__ int upper_bound_edges(const double *e, int n, double v)
{
    int lo = 0, hi = n;
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (e[mid] <= v) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// bytes of walker state in shared memory for a CTA of `block` threads
__host__ __device__ constexpr size_t walker_smem_bytes(int block) { return (size_t)block * 3 * sizeof(AxisF); }

// position of plane p (relative index) of axis a
template <int EDGE_MODE>
__device__ __forceinline__ double plane_pos(const MeshDev &m, const double *e, int a, int base, int p)
{
    if (EDGE_MODE == EDGES_ARITH) return fma((double)p, m.h[a], m.e0[a]);
    return e[base + p];
}

// Returns false if the ray is rejected by the box / direction rules of O1.  axf points at this thread's
// axis-0 record; axis a is at [a * stride].  `e` = the concatenated plane table (global or shared).
template <int EDGE_MODE>
__device__ __forceinline__ bool walker_init(Walker &w, AxisF *axf, int stride, const MeshDev &m, const double *e,
                                            const double o[3], const double d[3])
{
    const int base[3] = {0, m.nx + 1, m.nx + m.ny + 2};
    const int n[3] = {m.nx, m.ny, m.nz};
    const int dcell[3] = {1, m.nx, m.nx * m.ny};
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    int idx[3], pl[3], dc[3];
    double t[3];
    bool movable = false;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double lo = plane_pos<EDGE_MODE>(m, e, a, base[a], 0), hi = plane_pos<EDGE_MODE>(m, e, a, base[a], n[a]);
        if (!(o[a] >= lo && o[a] < hi)) return false;                          // half-open box (Q8)
        // O3: i = upper_bound(edges, o) - 1, by pure comparisons against the plane positions
        int l = 0, r = n[a] + 1;
        while (l < r) {
            const int mid = (l + r) >> 1;
            if (plane_pos<EDGE_MODE>(m, e, a, base[a], mid) <= o[a]) l = mid + 1; else r = mid;
        }
        idx[a] = l - 1;
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double dd = d[a];
        const double inv = (dd != 0.0) ? __drcp_rn(dd) : 0.0;
        if (dd == 0.0 || !isfinite(inv)) {                                     // Q10: the axis never steps
            pl[a] = idx[a] | (0xffff << 16);   // never selected; the low half keeps the axis' cell index (walker_cell_index)
            dc[a] = 0;
            axf[a * stride] = AxisF{o[a], 0.0};
            t[a] = inf;
        } else {
            movable = true;
            const bool up = dd > 0.0;
            const int p = up ? idx[a] + 1 : idx[a];
            pl[a] = p | ((up ? n[a] : 0) << 16);
            dc[a] = up ? dcell[a] : -dcell[a];
            axf[a * stride] = AxisF{o[a], inv};
            t[a] = __dmul_rn(__dsub_rn(plane_pos<EDGE_MODE>(m, e, a, base[a], p), o[a]), inv);   // O4
        }
    }
    w.t0 = t[0]; w.t1 = t[1]; w.t2 = t[2];
    w.pl0 = pl[0]; w.pl1 = pl[1]; w.pl2 = pl[2];
    w.dc0 = dc[0]; w.dc1 = dc[1]; w.dc2 = dc[2];
    w.tcur = 0.0;
    w.c = idx[0] + m.nx * (idx[1] + m.ny * idx[2]);
    return movable;
}

// Cell index along one axis from the walker's packed word: the next plane is i + 1 when stepping up, i when stepping
// down; an axis that never steps keeps i itself.
__device__ __forceinline__ int walker_cell_index(int pl, int dc) { return (pl & 0xffff) - (dc > 0 ? 1 : 0); }

// One step of the merge (O5).  On return `cell` = the cell just traversed, `len` its segment length;
// the return value is true when the ray has left the mesh.
// LIMIT (next-event walk): a pending crossing with parameter >= 1 ends the walk AT the detector (t = 1).
template <int EDGE_MODE, bool LIMIT = false>
__device__ __forceinline__ bool walker_step(Walker &w, const AxisF *axf, int stride, const MeshDev &m, const double *e,
                                            int &cell, double &len)
{
    const bool ysel = w.t1 < w.t0;                 // ties keep x
    const double tm = ysel ? w.t1 : w.t0;
    const bool zsel = w.t2 < tm;                   // ties keep x / y
    const double tn = zsel ? w.t2 : tm;
    if (LIMIT && tn >= 1.0) {
        len = __dsub_rn(1.0, w.tcur);
        cell = w.c;
        return true;
    }
    const int a = zsel ? 2 : (ysel ? 1 : 0);
    const AxisF af = axf[a * stride];
    const int pl = zsel ? w.pl2 : (ysel ? w.pl1 : w.pl0);
    const int dc = zsel ? w.dc2 : (ysel ? w.dc1 : w.dc0);
    len = __dsub_rn(tn, w.tcur);
    w.tcur = tn;
    cell = w.c;
    const int p = pl & 0xffff;
    const bool leave = (p == (int)((unsigned)pl >> 16));
    const int s = dc > 0 ? 1 : -1;
    w.c += dc;
    const int pq = leave ? p : p + s;              // never read outside the table
    const int base = (EDGE_MODE == EDGES_ARITH) ? 0 : (zsel ? m.nx + m.ny + 2 : (ysel ? m.nx + 1 : 0));
    const double tnew = __dmul_rn(__dsub_rn(plane_pos<EDGE_MODE>(m, e, a, base, pq), af.o), af.iv);
    const int pln = pl + s;
    w.t0 = (zsel || ysel) ? w.t0 : tnew;
    w.t1 = (!zsel && ysel) ? tnew : w.t1;
    w.t2 = zsel ? tnew : w.t2;
    w.pl0 = (zsel || ysel) ? w.pl0 : pln;
    w.pl1 = (!zsel && ysel) ? pln : w.pl1;
    w.pl2 = zsel ? pln : w.pl2;
    return leave;
}

// ------------------------------------------------------------------------------------------------
// S4: total cross section of a cell from its record and the ray's per-material sigma values.
// sig[m * stride] is sigma of material m for this thread (shared memory, conflict-free).
// ------------------------------------------------------------------------------------------------
// Interface of a record type (the kernel is a template over it):
//   reset()                      once per ray
//   load(recs, ids, K, c)        start fetching cell c's record (issued one step ahead of its use)
//   value()                      the fetched record of the cell last passed to load(), as a small value
//   sigma(value, sig, stride, K) Sigma_t of that cell
template <int LAYOUT> struct CellRec;

// where a cell's score goes: the contiguous fp64 tally, unless the record type keeps the accumulator inside the record
struct PlainTally {
    static constexpr bool kTiled = false;
    static constexpr bool kCoarse = false;
    static __device__ __forceinline__ double *tally_at(double *tally, const void *, int cell) { return tally + cell; }
};

template <> struct CellRec<LAYOUT_K1> : PlainTally {
    typedef uint2 Value;
    uint2 v;
    __device__ __forceinline__ void reset() {}
    __device__ __forceinline__ void load(const void *recs, const uint8_t *, int, int c) { v = ldg_u2(reinterpret_cast<const uint2 *>(recs) + c); }
    // through L1: for walks whose consecutive cells are neighbours in memory (radial steps on an R-Z mesh)
    __device__ __forceinline__ void load_cached(const void *recs, const uint8_t *, int, int c) { v = __ldg(reinterpret_cast<const uint2 *>(recs) + c); }
    __device__ __forceinline__ Value value() const { return v; }
    static __device__ __forceinline__ float sigma(const Value &v, const float *sig, int stride, int) { return __uint_as_float(v.x) * sig[v.y * stride]; }
};

// 8-byte K = 1 records fetched as 32-byte aligned GROUPS OF FOUR (cells 4j .. 4j+3: neighbours along the fastest axis) and
// kept in registers: on an R-Z mesh a ray's consecutive cells are mostly radial neighbours, so three steps out of four
// need no load (the R-Z kernel is bound by L2 requests: one atomic and one record load per segment).
struct QuadRecK1 : PlainTally {
    typedef uint2 Value;
    uint4 a, b;
    int tag;       // index of the resident group, -1: none
    int sel;       // which of the four the current cell is
    __device__ __forceinline__ void reset() { tag = -1; }
    __device__ __forceinline__ void load(const void *recs, const uint8_t *, int, int c)
    {
        sel = c & 3;
        if ((c >> 2) != tag) {
            tag = c >> 2;
            ldg_256(reinterpret_cast<const uint4 *>(recs) + 2 * (size_t)tag, a, b);
        }
    }
    __device__ __forceinline__ Value value() const
    {
        const uint4 h = (sel & 2) ? b : a;
        return (sel & 1) ? make_uint2(h.z, h.w) : make_uint2(h.x, h.y);
    }
    static __device__ __forceinline__ float sigma(const Value &v, const float *sig, int stride, int) { return __uint_as_float(v.x) * sig[v.y * stride]; }
};

// 16-byte records (K = 2, 3) are fetched as 32-byte aligned PAIRS (cells 2j, 2j+1: x neighbours) with one
// LDG.E.256 and the pair is kept in registers: a step in x that stays inside the pair (about a quarter of
// all steps on a mesh with square xy cells) needs no load at all.  The kernel is bound by per-request units
// (one per lane for an uncoalesced access), so every load not issued is time saved.
struct PairRec {
    uint4 a, b;
    int tag;       // index of the resident pair, -1: none
    bool odd;      // which half the current cell is
    __device__ __forceinline__ void reset() { tag = -1; }
    __device__ __forceinline__ void load(const void *recs, const uint8_t *, int, int c)
    {
        odd = c & 1;
        if ((c >> 1) != tag) {
            tag = c >> 1;
            ldg_256(reinterpret_cast<const uint4 *>(recs) + 2 * (size_t)tag, a, b);
        }
    }
    __device__ __forceinline__ uint4 value() const { return odd ? b : a; }
};
struct SingleRec {
    uint4 v;
    __device__ __forceinline__ void reset() {}
    __device__ __forceinline__ void load(const void *recs, const uint8_t *, int, int c) { v = ldg_u4(reinterpret_cast<const uint4 *>(recs) + c); }
    __device__ __forceinline__ void load_cached(const void *recs, const uint8_t *, int, int c) { v = __ldg(reinterpret_cast<const uint4 *>(recs) + c); }
    __device__ __forceinline__ uint4 value() const { return v; }
};
template <typename Fetch> struct RecK2 : Fetch, PlainTally {
    typedef uint4 Value;
    static __device__ __forceinline__ float sigma(const Value &v, const float *sig, int stride, int)
    {
        float s = __uint_as_float(v.x) * sig[(v.z & 0xffu) * stride];
        return fmaf(__uint_as_float(v.y), sig[((v.z >> 8) & 0xffu) * stride], s);
    }
};
template <typename Fetch> struct RecK3 : Fetch, PlainTally {
    typedef uint4 Value;
    static __device__ __forceinline__ float sigma(const Value &v, const float *sig, int stride, int)
    {
        float s = __uint_as_float(v.x) * sig[(v.w & 0xffu) * stride];
        s = fmaf(__uint_as_float(v.y), sig[((v.w >> 8) & 0xffu) * stride], s);
        return fmaf(__uint_as_float(v.z), sig[((v.w >> 16) & 0xffu) * stride], s);
    }
};
template <> struct CellRec<LAYOUT_K2> : RecK2<SingleRec> {};
template <> struct CellRec<LAYOUT_K3> : RecK3<SingleRec> {};
template <> struct CellRec<LAYOUT_K2P> : RecK2<PairRec> {};
template <> struct CellRec<LAYOUT_K3P> : RecK3<PairRec> {};
template <> struct CellRec<LAYOUT_K4> : PlainTally {
    struct Value { uint4 v; uint32_t ids; };
    Value q;
    __device__ __forceinline__ void reset() {}
    __device__ __forceinline__ void load(const void *recs, const uint8_t *, int, int c)
    {
        const uint4 *p = reinterpret_cast<const uint4 *>(recs) + 2 * (size_t)c;
        q.v = ldg_u4(p);
        q.ids = __ldg(reinterpret_cast<const uint32_t *>(p + 1));
    }
    __device__ __forceinline__ Value value() const { return q; }
    static __device__ __forceinline__ float sigma(const Value &q, const float *sig, int stride, int)
    {
        float s = __uint_as_float(q.v.x) * sig[(q.ids & 0xffu) * stride];
        s = fmaf(__uint_as_float(q.v.y), sig[((q.ids >> 8) & 0xffu) * stride], s);
        s = fmaf(__uint_as_float(q.v.z), sig[((q.ids >> 16) & 0xffu) * stride], s);
        return fmaf(__uint_as_float(q.v.w), sig[(q.ids >> 24) * stride], s);
    }
};
// LAYOUT_K4 with the score accumulator INSIDE the record (bytes 24..31 of the 32-byte record are spare): on a mesh far
// larger than L2 every segment costs one DRAM fetch for the record and another for the tally sector; with the
// accumulator in the record's own sector the RED that follows the load hits L2.  The whole record is
// read with one plain (coherent) 32-byte load -- not ld.global.nc: the sector is written by the REDs of this kernel.
// flush_fused_kernel moves the in-record sums into the contiguous tally whenever the tally is looked at.
// Few distinct records (a lattice of pins, a room of air and concrete): the records live in a shared-memory dictionary
// and the mesh holds a small index per cell in 32-byte tiles of (x, y) cells, kept in registers.  A step in x or
// y that stays inside the tile needs no global load (2-byte indices, 4 x 4 tiles): 0.29 loads per segment on the PWR-like mesh against 0.65 with
// record pairs -- the cast kernel is bound by L2 tag look-ups, one per request.
// BITS = index width: 16 (tiles of 4 x 4 cells, up to 1024 records), 8 (8 x 4, up to 256), 4 (8 x 8, up to 16).
//
// BITS = 4 (kPerEntry): with at most 16 distinct records a ray evaluates Sigma_t of EVERY dictionary entry once, right after
// S1 (same fmaf chain in slot order, so the values are those of the per-cell evaluation bit for bit), into its own
// shared-memory column; a step then costs one 4-byte shared load instead of the 16-byte record and K sigma reads.
template <int BITS> struct TiledRec : PlainTally {
    static constexpr bool kTiled = true;
    static constexpr bool kPerEntry = BITS == 4;
    static constexpr int kXs = BITS == 16 ? 2 : 3;     // log2 of the tile's x extent
    static constexpr int kYs = BITS == 4 ? 3 : 2;      // log2 of the tile's y extent
    typedef typename std::conditional<BITS == 4, float, uint4>::type Value;   // kPerEntry: Sigma_t itself
    uint4 a, b;
    int tag;       // resident tile, -1: none
    int e;         // entry of the current cell inside the tile: (iy & (ty - 1)) * tx + (ix & (tx - 1))
    __device__ __forceinline__ void reset() { tag = -1; }
    __device__ __forceinline__ void load_tiled(const uint4 *tiles, int ntx, int nty, int ix, int iy, int iz)
    {
        const int t = (ix >> kXs) + ntx * ((iy >> kYs) + nty * iz);
        e = ((iy & ((1 << kYs) - 1)) << kXs) | (ix & ((1 << kXs) - 1));
        if (t != tag) {
            tag = t;
            ldg_256(tiles + 2 * (size_t)t, a, b);
        }
    }
    __device__ __forceinline__ int entry() const       // dictionary index of the current cell
    {
        const int bit = e * BITS;
        const int r = bit >> 5;
        const uint32_t lo4 = (r & 2) ? ((r & 1) ? a.w : a.z) : ((r & 1) ? a.y : a.x);
        const uint32_t hi4 = (r & 2) ? ((r & 1) ? b.w : b.z) : ((r & 1) ? b.y : b.x);
        const uint32_t w = (r & 4) ? hi4 : lo4;
        return (int)((w >> (bit & 31)) & ((1u << BITS) - 1u));
    }
    // sig_e: the thread's column of per-entry Sigma_t values (kPerEntry only)
    __device__ __forceinline__ Value value(const uint4 *s_dict, const float *sig_e, int stride) const
    {
        if constexpr (kPerEntry) {
            float v = sig_e[entry() * stride];
            asm volatile("" : "+f"(v));        // read out of the resident tile BEFORE the next tile is requested (no register copy of the tile)
            return v;
        } else
            return s_dict[entry()];
    }
    // Sigma_t of a dictionary record (K = 3 encoding), slots added in order
    static __device__ __forceinline__ float sigma_rec(const uint4 &v, const float *sig, int stride, int K)
    {
        float s = __uint_as_float(v.x) * sig[(v.w & 0xffu) * stride];
        if (K > 1) s = fmaf(__uint_as_float(v.y), sig[((v.w >> 8) & 0xffu) * stride], s);
        if (K > 2) s = fmaf(__uint_as_float(v.z), sig[((v.w >> 16) & 0xffu) * stride], s);
        return s;
    }
    static __device__ __forceinline__ float sigma(const Value &v, const float *sig, int stride, int K)
    {
        if constexpr (kPerEntry) return v;
        else return sigma_rec(v, sig, stride, K);
    }
};
constexpr int kPerEntryMax = 16;   // dictionary entries of the kPerEntry path (TiledRec<4>)
template <typename Rec, typename = void> struct rec_per_entry { static constexpr bool value = false; };
template <typename Rec> struct rec_per_entry<Rec, typename std::enable_if<Rec::kPerEntry>::type> { static constexpr bool value = true; };

template <> struct CellRec<LAYOUT_K4F> {
    static constexpr bool kTiled = false;
    static constexpr bool kCoarse = false;
    struct Value { uint4 v; uint32_t ids; };
    Value q;
    __device__ __forceinline__ void reset() {}
    __device__ __forceinline__ void load(const void *recs, const uint8_t *, int, int c)
    {
        uint4 lo, hi;
        asm volatile("ld.global.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(lo.x), "=r"(lo.y), "=r"(lo.z), "=r"(lo.w), "=r"(hi.x), "=r"(hi.y), "=r"(hi.z), "=r"(hi.w)
                     : "l"(reinterpret_cast<const uint4 *>(recs) + 2 * (size_t)c));
        q.v = lo;
        q.ids = hi.x;
    }
    __device__ __forceinline__ Value value() const { return q; }
    static __device__ __forceinline__ float sigma(const Value &q, const float *sig, int stride, int)
    {
        float s = __uint_as_float(q.v.x) * sig[(q.ids & 0xffu) * stride];
        s = fmaf(__uint_as_float(q.v.y), sig[((q.ids >> 8) & 0xffu) * stride], s);
        s = fmaf(__uint_as_float(q.v.z), sig[((q.ids >> 16) & 0xffu) * stride], s);
        return fmaf(__uint_as_float(q.v.w), sig[(q.ids >> 24) * stride], s);
    }
    static __device__ __forceinline__ double *tally_at(double *, const void *recs, int cell)
    {
        return reinterpret_cast<double *>(reinterpret_cast<uintptr_t>(recs) + 32 * (size_t)cell + 24);
    }
};
// Block-constant compositions (a material map coarser than the tally mesh: the usual case when a fine tally mesh is
// laid over a geometry of larger bodies; config 4 assigns materials in 8^3-cell blocks): mr_load_materials finds the
// largest s such that every aligned block of 2^s cells per axis holds ONE record, and stores one LAYOUT_K4 record per
// block.  On a mesh far larger than L2 the per-cell records (4.3 GB at 512^3) cost a DRAM line per segment; the
// coarse table (8 MB at s = 3) stays in L2, and a step that stays inside the block needs no load at all.
template <> struct CellRec<LAYOUT_C4> : PlainTally {
    static constexpr bool kCoarse = true;
    struct Value { uint4 v; uint32_t ids; };
    Value q;
    int tag;       // resident block, -1: none
    __device__ __forceinline__ void reset() { tag = -1; }
    __device__ __forceinline__ void load_coarse(const void *crecs, int s, int cnx, int cny, int ix, int iy, int iz)
    {
        const int b = (ix >> s) + cnx * ((iy >> s) + cny * (iz >> s));
        if (b != tag) {
            tag = b;
            uint4 lo, hi;
            ldg_256(reinterpret_cast<const uint4 *>(crecs) + 2 * (size_t)b, lo, hi);
            q.v = lo;
            q.ids = hi.x;
        }
    }
    __device__ __forceinline__ Value value() const { return q; }
    static __device__ __forceinline__ float sigma(const Value &q, const float *sig, int stride, int)
    {
        float s = __uint_as_float(q.v.x) * sig[(q.ids & 0xffu) * stride];
        s = fmaf(__uint_as_float(q.v.y), sig[((q.ids >> 8) & 0xffu) * stride], s);
        s = fmaf(__uint_as_float(q.v.z), sig[((q.ids >> 16) & 0xffu) * stride], s);
        return fmaf(__uint_as_float(q.v.w), sig[(q.ids >> 24) * stride], s);
    }
};

template <> struct CellRec<LAYOUT_D8> : PlainTally {
    struct Value { float4 a, b; };
    Value q;
    __device__ __forceinline__ void reset() {}
    __device__ __forceinline__ void load(const void *recs, const uint8_t *, int, int c)
    {
        uint4 lo, hi;
        ldg_256(reinterpret_cast<const uint4 *>(recs) + 2 * (size_t)c, lo, hi);
        q.a = make_float4(__uint_as_float(lo.x), __uint_as_float(lo.y), __uint_as_float(lo.z), __uint_as_float(lo.w));
        q.b = make_float4(__uint_as_float(hi.x), __uint_as_float(hi.y), __uint_as_float(hi.z), __uint_as_float(hi.w));
    }
    __device__ __forceinline__ Value value() const { return q; }
    static __device__ __forceinline__ float sigma(const Value &q, const float *sig, int stride, int)
    {
        float s = q.a.x * sig[0];
        s = fmaf(q.a.y, sig[stride], s);
        s = fmaf(q.a.z, sig[2 * stride], s);
        s = fmaf(q.a.w, sig[3 * stride], s);
        s = fmaf(q.b.x, sig[4 * stride], s);
        s = fmaf(q.b.y, sig[5 * stride], s);
        s = fmaf(q.b.z, sig[6 * stride], s);
        return fmaf(q.b.w, sig[7 * stride], s);
    }
};

// DOUBLE mode, K <= 3: the whole record in one 32-byte load (the generic layout costs 2K uncoalesced loads per cell).
// An empty slot packs as r = 0, id = 0 and adds +0 in the same slot order, like the fp32 records.
template <> struct CellRec<LAYOUT_DK3> : PlainTally {
    struct Value { double r0, r1, r2; uint32_t ids; };
    Value q;
    __device__ __forceinline__ void reset() {}
    __device__ __forceinline__ void load(const void *recs, const uint8_t *, int, int c)
    {
        uint4 lo, hi;
        ldg_256(reinterpret_cast<const uint4 *>(recs) + 2 * (size_t)c, lo, hi);
        q.r0 = __hiloint2double((int)lo.y, (int)lo.x);
        q.r1 = __hiloint2double((int)lo.w, (int)lo.z);
        q.r2 = __hiloint2double((int)hi.y, (int)hi.x);
        q.ids = hi.z;
    }
    __device__ __forceinline__ Value value() const { return q; }
    static __device__ __forceinline__ double sigma(const Value &q, const double *sig, int stride, int)
    {
        double s = q.r0 * sig[(q.ids & 0xffu) * stride];
        s += q.r1 * sig[((q.ids >> 8) & 0xffu) * stride];
        s += q.r2 * sig[((q.ids >> 16) & 0xffu) * stride];
        return s;
    }
};

// Generic layout, either precision: nothing is prefetched, the slots are read in sigma().
template <typename Real> struct CellRecGeneric : PlainTally {
    struct Value { const Real *coef; const uint8_t *ids; };
    Value q;
    __device__ __forceinline__ void reset() {}
    __device__ __forceinline__ void load(const void *recs, const uint8_t *idp, int K, int c)
    {
        q.coef = reinterpret_cast<const Real *>(recs) + (size_t)c * K;
        q.ids = idp + (size_t)c * K;
    }
    __device__ __forceinline__ Value value() const { return q; }
    static __device__ __forceinline__ Real sigma(const Value &q, const Real *sig, int stride, int K)
    {
        Real s = 0;
        for (int k = 0; k < K; ++k) {
            const unsigned id = __ldg(q.ids + k);
            if (id != 0xffu) s += __ldg(q.coef + k) * sig[id * stride];
        }
        return s;
    }
};

// rec.load_cached(...) where the record type has one (the load goes through L1), else rec.load(...)
template <typename Rec>
__device__ __forceinline__ auto load_record_cached(Rec &rec, const void *recs, const uint8_t *ids, int K, int c, int)
    -> decltype(rec.load_cached(recs, ids, K, c), void())
{
    rec.load_cached(recs, ids, K, c);
}
template <typename Rec>
__device__ __forceinline__ void load_record_cached(Rec &rec, const void *recs, const uint8_t *ids, int K, int c, long)
{
    rec.load(recs, ids, K, c);
}

// ------------------------------------------------------------------------------------------------
// S5: the two factors of Eq. (4) for one segment, x = Sigma * len >= 0:
//     g  = (1 - exp(-x)) / Sigma   (-> len as x -> 0, reading Q12),     ex = exp(-x)
// from ONE polynomial.  -x = k ln2 + r, |r| <= ln2/2; p = expm1(r) = r + r^2 q(r), q = Taylor
// 1/2! + r/3! + ...; exp(-x) = 2^k (1 + p); 1 - exp(-x) = (1 - 2^k) - 2^k p (no cancellation:
// 2^k (1+p) <= 0.71 for k < 0).  For k = 0 (x <= ln2/2, the common case in thin cells) g needs no
// division at all: (1 - e^{-x})/Sigma = len * (p/r) = len * (1 + r q(r)), which is also exact at x = 0.
// The attenuation is carried as a running product of ex itself: 1 + expm1(-x) would lose all
// precision once x > ~37.
//   FULL  (double mode): q to 1/13!, error ~1e-16; the k < 0 branch divides.
//   !FULL (mixed mode) : q to 1/8!, error < 6e-10 (the fp32 cross sections carry ~1e-7); the
//                        k < 0 branch uses rcp.approx + 2 Newton steps (error ~1e-16).
// ------------------------------------------------------------------------------------------------
__constant__ double c_expq[12] = {
    1.0 / 6227020800.0, 1.0 / 479001600.0, 1.0 / 39916800.0, 1.0 / 3628800.0, 1.0 / 362880.0, 1.0 / 40320.0,
    1.0 / 5040.0, 1.0 / 720.0, 1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0, 0.5};

template <bool FULL, bool WARP_VOTE = true>
__device__ __forceinline__ void score_terms(double S, double len, double &g, double &ex)
{
    const double x = S * len;
    const bool thin = x <= 0.34657359027997264;
    // WARP_VOTE false (the R-Z kernel, measured 6.3 against 6.6 ms): every lane picks its own arm
    if (!FULL && (WARP_VOTE ? __all_sync(__activemask(), thin) : thin)) {
        // Mixed mode, EVERY lane of the warp in a thin cell (k = 0; 85 % of the warp-steps on the PWR-like mesh): the same
        // expressions as the k = 0 case of the general path below (bit-identical results), without its predicated-off
        // range reduction.  The vote only picks the cheaper instruction stream: a warp with one thick cell takes the
        // general path for all its lanes instead of both arms one after the other.
        const double r = -x;
        double q = c_expq[5];
#pragma unroll
        for (int i = 6; i < 12; ++i) q = fma(q, r, c_expq[i]);
        ex = 1.0 + fma(r * r, q, r);
        g = fma(len * r, q, len);
        return;
    }
    double r = -x;
    int k = 0;
    if (x > 0.34657359027997264) {                                   // ln2 / 2
        const double kf = rint(x * -1.4426950408889634074);          // k = round(-x / ln2) < 0
        r = fma(kf, -6.93147180369123816490e-01, -x);                // Cody-Waite: ln2 = hi + lo
        r = fma(kf, -1.90821492927058770002e-10, r);
        k = (int)kf;                                                 // saturates for huge x
    }
    constexpr int first = FULL ? 0 : 5;
    double q = c_expq[first];
#pragma unroll
    for (int i = first + 1; i < 12; ++i) q = fma(q, r, c_expq[i]);
    const double p = fma(r * r, q, r);                               // expm1(r)
    if (k == 0) {
        ex = 1.0 + p;
        g = fma(len * r, q, len);                                    // len * (1 + r q)
    } else if (k >= -1022) {
        const double scale = __longlong_as_double((long long)(k + 1023) << 52);   // 2^k
        ex = fma(scale, p, scale);
        const double omex = fma(-scale, p, 1.0 - scale);
        if (FULL) {
            g = omex / S;
        } else {
            double y;
            asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(S));
            double err = fma(-S, y, 1.0);
            y = fma(y, err, y);
            err = fma(-S, y, 1.0);
            y = fma(y, err, y);
            g = omex * y;
        }
    } else {                                                         // x > 708: exp(-x) < 2.3e-308, flushed
        ex = 0.0;
        g = 1.0 / S;
    }
}

// ------------------------------------------------------------------------------------------------
// The cast kernel: one thread per ray (S1 -> S6).
//   dynamic shared memory: [edges: nedges doubles (EDGES_SHARED only)] [walker: 3 x blockDim x 16 B]
//                          [sigma: M x blockDim Real]
// ------------------------------------------------------------------------------------------------
__host__ __device__ constexpr size_t edges_smem_bytes_for(int nedges) { return sizeof(double) * (size_t)((nedges + 1) & ~1); }

template <typename Real, typename Rec, int EDGE_MODE>
__global__ void __launch_bounds__(256) cast_kernel(const __grid_constant__ CastParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int stride = blockDim.x;
    unsigned char *sp = smem_raw;
    double *s_edges = reinterpret_cast<double *>(sp);
    if (EDGE_MODE == EDGES_SHARED) sp += edges_smem_bytes_for(P.mesh.nedges);
    AxisF *axf = reinterpret_cast<AxisF *>(sp) + threadIdx.x;
    sp += sizeof(AxisF) * 3 * stride;
    Real *sig = reinterpret_cast<Real *>(sp) + threadIdx.x;
    sp += sizeof(Real) * (size_t)(P.M + P.N) * stride;
    constexpr bool kPerEntry = rec_per_entry<Rec>::value;
    Real *sig_e = reinterpret_cast<Real *>(sp) + threadIdx.x;   // kPerEntry: Sigma_t of every dictionary entry for this thread's ray
    if (kPerEntry) sp += sizeof(Real) * (size_t)kPerEntryMax * stride;
    uint4 *s_dict = reinterpret_cast<uint4 *>(sp);
    const double *e = (EDGE_MODE == EDGES_SHARED) ? s_edges : P.mesh.edges;
    if (EDGE_MODE == EDGES_SHARED) {
        for (int i = threadIdx.x; i < P.mesh.nedges; i += blockDim.x) s_edges[i] = __ldg(P.mesh.edges + i);
    }
    if (Rec::kTiled) {
        for (int i = threadIdx.x; i < P.ndict; i += blockDim.x) s_dict[i] = __ldg(P.dict + i);
    }
    if (EDGE_MODE == EDGES_SHARED || Rec::kTiled) __syncthreads();

    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned nseg = 0;
    bool accepted = false, live = i < P.n;
    if (live) {
        const long long r = P.perm ? (long long)__ldg(P.perm + i) : i;
        const Ray<Real> R = load_ray<Real>(P.rays, r);
        Walker w;
        accepted = R.finite && (R.E > (Real)0) && walker_init<EDGE_MODE>(w, axf, stride, P.mesh, e, R.o, R.d);
        if (accepted) {
            // S1: every material's sigma at the ray's energy, kept in this thread's shared column
            sigma_all<Real>(P.xs, P.M, P.N, P.mix_off, P.mix_nuc, P.mix_w, R.E, sig, stride);
            if constexpr (kPerEntry)
                for (int q = 0; q < P.ndict; ++q) sig_e[q * stride] = Rec::sigma_rec(s_dict[q], sig, stride, P.K);

            double wa = R.W;   // W * exp(-tau), a running product of exp(-x)
            double *const tally = P.tally;
            // S4 + S5 + S6 for one segment: score = W e^{-tau} (1 - e^{-x}) / Sigma, x = Sigma * len (Eq. (4));
            // a zero-length segment scores exactly 0: nothing to add
            auto score = [&](const typename Rec::Value &cur, int cell, double len, const bool aggregate) {
                const double S = (double)Rec::sigma(cur, sig, stride, P.K);
                double g, ex;
                score_terms<sizeof(Real) == 8>(S, len, g, ex);
                double v = wa * g;
                bool add = len > 0.0;
                // Warp-aggregated atomics for the first P.agg_first segments of a ray: rays born in one small region (a
                // source volume of a few cells) hit the same cells in their first steps, and same-address REDs serialise
                // in L2.  Lanes of the warp that score into the same cell are found with match.any; the lowest adds the sum.
                if (aggregate) {
                    const unsigned act = __activemask();
                    const unsigned peers = __match_any_sync(act, add ? cell : -1 - (int)(threadIdx.x & 31));
                    if (peers & (peers - 1)) {                       // somebody shares this cell
                        const int me = threadIdx.x & 31, leader = __ffs(peers) - 1;
                        double sum = 0.0;
                        for (unsigned rest = peers; rest; rest &= rest - 1) sum += __shfl_sync(peers, v, __ffs(rest) - 1);
                        v = sum;
                        add = add && me == leader;
                    }
                }
                if (add) red_add_f64(Rec::tally_at(tally, P.recs, cell), v);
                wa *= ex;
                ++nseg;
            };
            Rec rec;
            rec.reset();
            // the record (or index tile) of the cell the walker stands in
            auto fetch = [&]() {
                if constexpr (Rec::kTiled)
                    rec.load_tiled(P.tiles, P.ntx, P.nty, walker_cell_index(w.pl0, w.dc0), walker_cell_index(w.pl1, w.dc1),
                                   walker_cell_index(w.pl2, w.dc2));
                else if constexpr (Rec::kCoarse)
                    rec.load_coarse(P.crecs, P.cshift, P.cnx, P.cny, walker_cell_index(w.pl0, w.dc0),
                                    walker_cell_index(w.pl1, w.dc1), walker_cell_index(w.pl2, w.dc2));
                else
                    rec.load(P.recs, P.ids, P.K, w.c);
            };
            fetch();
            // one segment; returns true when the ray has left the mesh
            auto segment = [&](const bool aggregate) {
                int cell;
                double len;
                const bool leave = walker_step<EDGE_MODE>(w, axf, stride, P.mesh, e, cell, len);
                typename Rec::Value cur;
                if constexpr (Rec::kTiled) cur = rec.value(s_dict, (const float *)sig_e, stride);
                else cur = rec.value();
                if (!leave) fetch();                              // next cell's record: in flight during the score
                score(cur, cell, len, aggregate);
                return leave;
            };
            // the first P.agg_first segments with warp-aggregated atomics, the rest (the hot loop) without the test
            bool left = false;
            for (int k = 0; k < P.agg_first && !left; ++k) left = segment(true);
            while (!left) left = segment(false);
        }
    }
    // per-warp totals -> three global counters
    const unsigned full = 0xffffffffu;
    const unsigned acc = __popc(__ballot_sync(full, accepted));
    const unsigned rej = __popc(__ballot_sync(full, live && !accepted));
    unsigned long long segs = nseg;
    for (int o = 16; o > 0; o >>= 1) segs += __shfl_xor_sync(full, segs, o);
    if ((threadIdx.x & 31) == 0) {
        if (acc) atomicAdd(P.counters + 0, (unsigned long long)acc);
        if (rej) atomicAdd(P.counters + 1, (unsigned long long)rej);
        if (segs) atomicAdd(P.counters + 2, segs);
    }
}

// ------------------------------------------------------------------------------------------------
// The cast kernel with COOPERATIVE tally adds (north_star subsystem (4); option MR_OPT_COOP_FLUSH).
//
// cast_kernel issues one red.global.add.f64 per segment from lanes that are 32 unrelated rays: 32 sectors per
// instruction, and the L2 atomic unit takes about 2.1e11 such sector-requests per second (mr_microbench_red) -- the
// unit the kernel saturates.  The same unit takes twice as many lane-adds when pairs of lanes share a sector.  Lanes of
// different rays never do; CONSECUTIVE segments of one ray often do (an x-step stays inside the 32-byte sector of four
// cells three times out of four).  So every lane walks kCoopWindow steps, staging (cell, score) in its own
// shared-memory column; then the warp adds the staged pairs TRANSPOSED: one instruction carries the kCoopWindow
// consecutive segments of 32 / kCoopWindow rays.  Scores, cells and their order per ray are unchanged; tally[c]
// receives the same values in another order (reading Q18).
//   column layout: entry (lane, row) at lane * (kCoopWindow + 1) + row -- conflict-free for the lane-wise writes
//   (9 is odd) and nearly so for the transposed reads.
//   dynamic shared memory: as cast_kernel, then per warp 32 x 9 x (8 + 4) bytes.
// ------------------------------------------------------------------------------------------------
constexpr int kCoopWindow = 8;
__host__ __device__ constexpr size_t coop_warp_smem_bytes() { return (size_t)32 * (kCoopWindow + 1) * 12; }

// PAIR: instead of the 8-step shared-memory staging, every lane walks TWO steps and exchanges one (cell, score) pair with its
// neighbour lane by shuffles, so that lanes 2i and 2i+1 of an add instruction carry two consecutive segments of one ray
// (the same 128-byte tally line for 15 of 16 x-steps): fewer L2 requests than segments at 3 shuffles and a few selects per
// two segments, no shared memory.
template <typename Real, typename Rec, int EDGE_MODE, bool PAIR = false>
__global__ void __launch_bounds__(256) cast_coop_kernel(const __grid_constant__ CastParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int stride = blockDim.x;
    unsigned char *sp = smem_raw;
    double *s_edges = reinterpret_cast<double *>(sp);
    if (EDGE_MODE == EDGES_SHARED) sp += edges_smem_bytes_for(P.mesh.nedges);
    AxisF *axf = reinterpret_cast<AxisF *>(sp) + threadIdx.x;
    sp += sizeof(AxisF) * 3 * stride;
    Real *sig = reinterpret_cast<Real *>(sp) + threadIdx.x;
    sp += (sizeof(Real) * (size_t)(P.M + P.N) * stride + 15) & ~(size_t)15;
    constexpr bool kPerEntry = rec_per_entry<Rec>::value;
    Real *sig_e = reinterpret_cast<Real *>(sp) + threadIdx.x;
    if (kPerEntry) sp += sizeof(Real) * (size_t)kPerEntryMax * stride;
    uint4 *s_dict = reinterpret_cast<uint4 *>(sp);
    if (Rec::kTiled) sp += sizeof(uint4) * (size_t)P.ndict;
    double *c_score = reinterpret_cast<double *>(sp + (threadIdx.x >> 5) * coop_warp_smem_bytes());
    unsigned *c_cell = reinterpret_cast<unsigned *>(c_score + 32 * (kCoopWindow + 1));
    const double *e = (EDGE_MODE == EDGES_SHARED) ? s_edges : P.mesh.edges;
    if (EDGE_MODE == EDGES_SHARED) {
        for (int i = threadIdx.x; i < P.mesh.nedges; i += blockDim.x) s_edges[i] = __ldg(P.mesh.edges + i);
    }
    if (Rec::kTiled) {
        for (int i = threadIdx.x; i < P.ndict; i += blockDim.x) s_dict[i] = __ldg(P.dict + i);
    }
    if (EDGE_MODE == EDGES_SHARED || Rec::kTiled) __syncthreads();

    const unsigned full = 0xffffffffu;
    const unsigned lane = threadIdx.x & 31;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = i < P.n;
    bool accepted = false;
    unsigned nseg = 0;
    Walker w{};
    Rec rec;
    double wa = 0.0;
    auto fetch = [&]() {
        if constexpr (Rec::kTiled)
            rec.load_tiled(P.tiles, P.ntx, P.nty, walker_cell_index(w.pl0, w.dc0), walker_cell_index(w.pl1, w.dc1),
                           walker_cell_index(w.pl2, w.dc2));
        else if constexpr (Rec::kCoarse)
            rec.load_coarse(P.crecs, P.cshift, P.cnx, P.cny, walker_cell_index(w.pl0, w.dc0), walker_cell_index(w.pl1, w.dc1),
                            walker_cell_index(w.pl2, w.dc2));
        else
            rec.load(P.recs, P.ids, P.K, w.c);
    };
    if (live) {
        const long long r = P.perm ? (long long)__ldg(P.perm + i) : i;
        const Ray<Real> R = load_ray<Real>(P.rays, r);
        accepted = R.finite && (R.E > (Real)0) && walker_init<EDGE_MODE>(w, axf, stride, P.mesh, e, R.o, R.d);
        if (accepted) {
            sigma_all<Real>(P.xs, P.M, P.N, P.mix_off, P.mix_nuc, P.mix_w, R.E, sig, stride);
            if constexpr (kPerEntry)
                for (int q = 0; q < P.ndict; ++q) sig_e[q * stride] = Rec::sigma_rec(s_dict[q], sig, stride, P.K);
            wa = R.W;
            rec.reset();
            fetch();
        }
    }
    bool left = !accepted;
    // one segment: walk, record, Eq. (4); returns the score (0 for a zero-length segment) and the cell
    auto segment = [&](int &cell, double &v) {
        double len;
        const bool leave = walker_step<EDGE_MODE>(w, axf, stride, P.mesh, e, cell, len);
        typename Rec::Value cur;
        if constexpr (Rec::kTiled) cur = rec.value(s_dict, (const float *)sig_e, stride);
        else cur = rec.value();
        if (!leave) fetch();
        const double S = (double)Rec::sigma(cur, sig, stride, P.K);
        double g, ex;
        score_terms<sizeof(Real) == 8>(S, len, g, ex);
        v = wa * g;
        wa *= ex;
        ++nseg;
        left = leave;
        return len > 0.0;
    };
    // the first P.agg_first segments of a ray with warp-aggregated atomics (rays born in one small region, §4.7)
    for (int k = 0; k < P.agg_first; ++k) {
        if (!left) {
            int cell;
            double v;
            bool add = segment(cell, v);
            const unsigned act = __activemask();
            const unsigned peers = __match_any_sync(act, add ? cell : -1 - (int)lane);
            if (peers & (peers - 1)) {
                const int leader = __ffs(peers) - 1;
                double sum = 0.0;
                for (unsigned rest = peers; rest; rest &= rest - 1) sum += __shfl_sync(peers, v, __ffs(rest) - 1);
                v = sum;
                add = add && (int)lane == leader;
            }
            if (add) red_add_f64(P.tally + cell, v);
        }
    }
    if (PAIR) {
        const bool even = !(lane & 1);
        while (__any_sync(full, !left)) {
            int cA = -1, cB = -1;                      // -1: nothing to add (zero-length segment, finished ray)
            double vA = 0.0, vB = 0.0;
            if (!left) {
                int cell;
                if (segment(cell, vA)) cA = cell;
            }
            if (!left) {
                int cell;
                if (segment(cell, vB)) cB = cell;
            }
            const int gc = even ? cB : cA;
            const double gv = even ? vB : vA;
            const int rc = __shfl_xor_sync(full, gc, 1);
            const double rv = __shfl_xor_sync(full, gv, 1);
            const int c1 = even ? cA : rc, c2 = even ? rc : cB;       // instruction 1: ray 2i's A and B; instruction 2: ray 2i+1's
            const double v1 = even ? vA : rv, v2 = even ? rv : vB;
            if (c1 >= 0) red_add_f64(P.tally + c1, v1);
            if (c2 >= 0) red_add_f64(P.tally + c2, v2);
        }
    } else
    // windows of kCoopWindow steps, then the transposed adds
    while (__any_sync(full, !left)) {
        int k = 0;
#pragma unroll 1
        for (int j = 0; j < kCoopWindow; ++j) {
            if (!left) {
                int cell;
                double v;
                if (segment(cell, v)) {
                    c_cell[lane * (kCoopWindow + 1) + k] = (unsigned)cell;
                    c_score[lane * (kCoopWindow + 1) + k] = v;
                    ++k;
                }
            }
        }
        __syncwarp();
        const int row = lane % kCoopWindow;
#pragma unroll
        for (int p = 0; p < kCoopWindow; ++p) {
            const int src = p * (32 / kCoopWindow) + lane / kCoopWindow;
            const int kk = __shfl_sync(full, k, src);
            if (row < kk) red_add_f64(P.tally + c_cell[src * (kCoopWindow + 1) + row], c_score[src * (kCoopWindow + 1) + row]);
        }
        __syncwarp();
    }
    const unsigned acc = __popc(__ballot_sync(full, accepted));
    const unsigned rej = __popc(__ballot_sync(full, live && !accepted));
    unsigned long long segs = nseg;
    for (int o = 16; o > 0; o >>= 1) segs += __shfl_xor_sync(full, segs, o);
    if (lane == 0) {
        if (acc) atomicAdd(P.counters + 0, (unsigned long long)acc);
        if (rej) atomicAdd(P.counters + 1, (unsigned long long)rej);
        if (segs) atomicAdd(P.counters + 2, segs);
    }
}

// ------------------------------------------------------------------------------------------------
// The trace kernel (test entry point mr_trace_rays): the same walker, no cross sections, no tally.
//   dynamic shared memory: [edges (EDGES_SHARED only)] [walker: 3 x blockDim x 16 B]
// ------------------------------------------------------------------------------------------------
template <int EDGE_MODE>
__global__ void __launch_bounds__(256) trace_kernel(const __grid_constant__ TraceParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int stride = blockDim.x;
    unsigned char *sp = smem_raw;
    double *s_edges = reinterpret_cast<double *>(sp);
    if (EDGE_MODE == EDGES_SHARED) sp += edges_smem_bytes_for(P.mesh.nedges);
    AxisF *axf = reinterpret_cast<AxisF *>(sp) + threadIdx.x;
    const double *e = (EDGE_MODE == EDGES_SHARED) ? s_edges : P.mesh.edges;
    if (EDGE_MODE == EDGES_SHARED) {
        for (int i = threadIdx.x; i < P.mesh.nedges; i += blockDim.x) s_edges[i] = __ldg(P.mesh.edges + i);
        __syncthreads();
    }
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= P.n) return;
    double o[3], d[3];
    bool ok;
    if (P.ray_is_double) {
        const Ray<double> R = load_ray_f64(P.rays, r);
        for (int a = 0; a < 3; ++a) { o[a] = R.o[a]; d[a] = R.d[a]; }
        ok = R.finite && R.E > 0.0;
    } else {
        const Ray<float> R = load_ray_f32(P.rays, r);
        for (int a = 0; a < 3; ++a) { o[a] = R.o[a]; d[a] = R.d[a]; }
        ok = R.finite && R.E > 0.0f;
    }
    Walker w;
    ok = ok && walker_init<EDGE_MODE>(w, axf, stride, P.mesh, e, o, d);
    unsigned nseg = 0;
    unsigned long long h = 0;
    if (ok) {
        h = 0xcbf29ce484222325ULL;
        for (;;) {
            int cell;
            double len;
            const bool leave = walker_step<EDGE_MODE>(w, axf, stride, P.mesh, e, cell, len);
            if ((long long)nseg < P.cap) {
                if (P.cells) P.cells[r * P.cap + nseg] = cell;
                if (P.lens) P.lens[r * P.cap + nseg] = len;
            }
            const unsigned cu = (unsigned)cell;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                h ^= (unsigned long long)((cu >> (8 * b)) & 0xffu);
                h *= 0x100000001b3ULL;
            }
            ++nseg;
            if (leave) break;
        }
    }
    if (P.nseg) P.nseg[r] = nseg;
    if (P.hash) P.hash[r] = h;
}

// ------------------------------------------------------------------------------------------------
// R-Z (2-D cylindrical) tally mesh, SURVEY.md §8(f) NEXT-4.  Cell (ir, iz), c = ir + nr*iz, radii
// re[0] = 0 < ... < re[nr], planes ze[0..nz]; MeshDev carries nx = nr, ny = 1, nz and edges = re | (1 pad) | ze laid
// out like a Cartesian mesh with ny = 1 (x planes = radii, z planes = ze).  Steps Z1-Z5 of DESIGN.md §10.6, every
// trace-determining operation written with a rounding-explicit intrinsic (no contraction):
//   rho0^2 = ox*ox + oy*oy,  a = dx*dx + dy*dy,  b = ox*dx + oy*dy,  inv_a = 1/a
//   cylinder p:  cc = rho0^2 - r_p*r_p,  D = b*b - a*cc,  t_in/out = max(0, (-b -/+ sqrt(D)) * inv_a)
//   plane p:     t_z = (z_p - oz) * (1/dz);  ties: radial before axial
// One thread per ray; TRACE = the test entry (per-ray count / hash / lists, no cross sections, no tally).
//   dynamic shared memory: [edges] [sigma: (M+N) x blockDim Real]
// ------------------------------------------------------------------------------------------------
struct RzParams {
    CastParams c;            // mesh (nx = nr, ny = 1), records, tables, rays, tally, counters
    uint32_t *nseg;          // TRACE outputs, any may be null
    unsigned long long *hash;
    int32_t *cells;
    double *lens;
    long long cap;
    int ray_is_double;
    int spherical;           // 1: 1-D spherical shells about the origin (no axial crossings; nz = 1)
};

__device__ __forceinline__ double rz_t_radial(double b, double a, double inv_a, double rho2, double rp, bool outward)
{
    const double cc = __dsub_rn(rho2, __dmul_rn(rp, rp));
    const double D = __dsub_rn(__dmul_rn(b, b), __dmul_rn(a, cc));
    const double sq = __dsqrt_rn(D);
    const double num = outward ? __dadd_rn(-b, sq) : __dsub_rn(-b, sq);
    return fmax(0.0, __dmul_rn(num, inv_a));
}

// Ray lengths on these meshes vary by about 2x around their mean (17.8 of 32 lanes were active with one ray per
// thread, and ordering the rays by length makes neighbouring lanes hammer the same ring-shaped cells), so the kernel
// is PERSISTENT: a lane that finishes its ray takes the next one from a global counter (P.counters[3], zeroed before
// the launch); refills are batched (at least kRefillLanes idle lanes, or nothing left to do) to keep the divergent
// per-ray set-up rare.
constexpr int kRefillLanes = 8;

// squares of the radii, kept beside the radii in shared memory (r_p * r_p rounded once: the value every D_p is formed from)
__host__ __device__ constexpr size_t rz_re2_bytes(int nr) { return sizeof(double) * (size_t)((nr + 2) & ~1); }

__device__ __forceinline__ double lds_f64(unsigned addr)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

// D_p = b*b - a*(rho0^2 - r_p^2), every operation rounded to nearest (Z4); r2 = r_p * r_p
__device__ __forceinline__ double rz_disc(double bb, double a, double rho2, double r2)
{
    return __dsub_rn(bb, __dmul_rn(a, __dsub_rn(rho2, r2)));
}

//   dynamic shared memory: [edges] [r_p^2: nr + 1 doubles] [sigma: (M+N) x blockDim Real] [cast: per warp 32 x 9 staged pairs]
template <typename Real, typename Rec, bool TRACE>
__global__ void __launch_bounds__(256, 3) rz_kernel(const __grid_constant__ RzParams Q)
{
    const CastParams &P = Q.c;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int stride = blockDim.x;
    const int nr = P.mesh.nx, nz = P.mesh.nz;
    double *s_edges = reinterpret_cast<double *>(smem_raw);
    double *s_re2 = reinterpret_cast<double *>(smem_raw + edges_smem_bytes_for(P.mesh.nedges));
    unsigned char *sp = smem_raw + edges_smem_bytes_for(P.mesh.nedges) + rz_re2_bytes(nr);
    Real *sig = reinterpret_cast<Real *>(sp) + threadIdx.x;
    // cast launches only: per warp 32 x 9 staged (score, cell) pairs behind the sigma columns
    unsigned char *stage = sp + ((sizeof(Real) * (size_t)(P.M + P.N) * stride + 15) & ~(size_t)15);
    double *c_score = reinterpret_cast<double *>(stage + (threadIdx.x >> 5) * coop_warp_smem_bytes());
    unsigned *c_cell = reinterpret_cast<unsigned *>(c_score + 32 * (kCoopWindow + 1));
    for (int i = threadIdx.x; i < P.mesh.nedges; i += blockDim.x) {
        const double v = __ldg(P.mesh.edges + i);
        s_edges[i] = v;
        if (i <= nr) s_re2[i] = __dmul_rn(v, v);
    }
    __syncthreads();
    const double *re2 = s_re2, *ze = s_edges + nr + 3;        // Cartesian layout with ny = 1: x | y (2 planes) | z
    const unsigned re2_addr = (unsigned)__cvta_generic_to_shared(s_re2), ze_addr = (unsigned)__cvta_generic_to_shared(ze);
    const bool sph = Q.spherical != 0;
    const unsigned full = 0xffffffffu;
    const unsigned lane = threadIdx.x & 31;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);

    // per-lane ray state
    long long r = -1;
    bool active = false, inward = false;
    double oz = 0.0, rho2 = 0.0, a = 0.0, b = 0.0, bb = 0.0, inv_a = 0.0, inv_z = 0.0, t_r = inf, t_z = inf, t_cur = 0.0, wa = 0.0;
    int ir = 0, iz = 0, pz = 0, stepz = 0;
    int i_turn = 1;          // innermost cylinder the ray crosses: D_p > 0 exactly for p >= i_turn (D_p is non-decreasing in p)
    unsigned nseg = 0;
    unsigned long long h = 0;
    Rec rec;
    // per-lane totals for the counters
    unsigned n_acc = 0, n_rej = 0;
    unsigned long long n_seg = 0;
    bool exhausted = false;                                     // warp-uniform: the ray counter has run past P.n

    for (;;) {
        const unsigned idle = __ballot_sync(full, !active);
        if (!exhausted && idle && (__popc(idle) >= kRefillLanes || idle == full)) {
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(P.counters + 3, (unsigned long long)__popc(idle));
            base = __shfl_sync(full, base, 0);
            exhausted = (long long)(base + __popc(idle)) >= P.n;
            if (!active) {
                r = (long long)base + __popc(idle & ((1u << lane) - 1u));
                if (r < P.n) {
                    double ox, oy, dx, dy, dz, W;
                    Real E;
                    bool fin;
                    if (sizeof(Real) == 8 || (TRACE && Q.ray_is_double)) {
                        const Ray<double> R = load_ray_f64(P.rays, r);
                        ox = R.o[0]; oy = R.o[1]; oz = R.o[2]; dx = R.d[0]; dy = R.d[1]; dz = R.d[2]; W = R.W; E = (Real)R.E; fin = R.finite && R.E > 0.0;
                    } else {
                        const Ray<float> R = load_ray_f32(P.rays, r);
                        ox = R.o[0]; oy = R.o[1]; oz = R.o[2]; dx = R.d[0]; dy = R.d[1]; dz = R.d[2]; W = R.W; E = (Real)R.E; fin = R.finite && R.E > 0.0f;
                    }
                    // Z1
                    rho2 = __dadd_rn(__dmul_rn(ox, ox), __dmul_rn(oy, oy));
                    a = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
                    if (sph) {
                        rho2 = __dadd_rn(rho2, __dmul_rn(oz, oz));
                        a = __dadd_rn(a, __dmul_rn(dz, dz));
                    }
                    inv_a = (a != 0.0) ? __drcp_rn(a) : 0.0;
                    const bool radial = (a != 0.0) && isfinite(inv_a) && isfinite(a);
                    inv_z = (dz != 0.0) ? __drcp_rn(dz) : 0.0;
                    const bool axial = !sph && (dz != 0.0) && isfinite(inv_z);
                    const bool accepted = fin && (radial || axial) && (rho2 < re2[nr]) && (sph || (oz >= ze[0] && oz < ze[nz]));
                    nseg = 0;
                    h = 0;
                    if (accepted) {
                        if (!TRACE) sigma_all<Real>(P.xs, P.M, P.N, P.mix_off, P.mix_nuc, P.mix_w, E, sig, stride);   // Z2
                        // Z3: ir = #{p : r_p^2 <= rho0^2} - 1 (r_p^2 is non-decreasing in p), iz by comparisons
                        int lo = 0, hi = nr + 1;
                        while (lo < hi) {
                            const int mid = (lo + hi) >> 1;
                            if (re2[mid] <= rho2) lo = mid + 1; else hi = mid;
                        }
                        ir = lo - 1;
                        iz = sph ? 0 : upper_bound_edges(ze, nz + 1, oz) - 1;
                        // Z4
                        b = __dadd_rn(__dmul_rn(ox, dx), __dmul_rn(oy, dy));
                        if (sph) b = __dadd_rn(b, __dmul_rn(oz, dz));
                        bb = __dmul_rn(b, b);
                        inward = false;
                        i_turn = ir + 1;
                        t_r = inf; t_z = inf; t_cur = 0.0; pz = 0; stepz = 0;
                        if (radial) {
                            if (b < 0.0 && ir >= 1) {
                                // The walk asks "D_p > 0 ?" of every inner cylinder it comes to.  D_p is a non-decreasing function of p
                                // (r_p^2 is, and every operation of rz_disc is monotone under round-to-nearest), so the answers are
                                // known from ONE index, found here by bisection with the walk's own expression: the decisions are
                                // those of Z4 bit for bit, and a step evaluates the discriminant of one cylinder only.
                                int l = 1, u = ir + 1;
                                while (l < u) {
                                    const int mid = (l + u) >> 1;
                                    if (rz_disc(bb, a, rho2, re2[mid]) > 0.0) u = mid; else l = mid + 1;
                                }
                                i_turn = l;
                                inward = ir >= i_turn;
                            }
                            const double D = rz_disc(bb, a, rho2, re2[inward ? ir : ir + 1]);
                            const double sq = __dsqrt_rn(D);
                            t_r = fmax(0.0, __dmul_rn(inward ? __dsub_rn(-b, sq) : __dadd_rn(-b, sq), inv_a));
                        }
                        if (axial) {
                            stepz = dz > 0.0 ? 1 : -1;
                            pz = dz > 0.0 ? iz + 1 : iz;
                            t_z = __dmul_rn(__dsub_rn(ze[pz], oz), inv_z);
                        }
                        if (TRACE) h = 0xcbf29ce484222325ULL;
                        wa = W;
                        if (!TRACE) {
                            rec.reset();
                            rec.load(P.recs, P.ids, P.K, ir + nr * iz);
                        }
                        active = true;
                        ++n_acc;
                    } else {
                        ++n_rej;
                        if (TRACE) {
                            if (Q.nseg) Q.nseg[r] = 0;
                            if (Q.hash) Q.hash[r] = 0;
                        }
                    }
                }
            }
        }
        if (__ballot_sync(full, active) == 0) {
            if (exhausted) break;
            continue;
        }
        // kCoopWindow steps per lane, every scored segment staged in the lane's shared-memory column, then the warp adds
        // the staged pairs TRANSPOSED: one instruction carries 8 consecutive segments of each of 4 rays.  On an R-Z mesh
        // consecutive cells of a ray are mostly radial neighbours, i.e. neighbours in the tally: 4 of them share a 32-byte
        // sector, and the L2 request rate (1 atomic + 1 record load per segment) is what bounds this kernel.
        int k = 0;
        double *st_score = c_score + lane * (kCoopWindow + 1);
        unsigned *st_cell = c_cell + lane * (kCoopWindow + 1);
#pragma unroll 1
        for (int j = 0; j < (TRACE ? 1 : kCoopWindow); ++j)
        if (active) {
            // Z5: one segment
            const bool ax = t_z < t_r;                      // ties: radial first
            const double tn = ax ? t_z : t_r;
            const double len = __dsub_rn(tn, t_cur);
            const int cell = ir + nr * iz;
            const int iz_n = ax ? iz + stepz : iz;
            const int ir_n = ax ? ir : (inward ? ir - 1 : ir + 1);
            const bool out = iz_n < 0 || iz_n >= nz || ir_n >= nr;      // the ray leaves the mesh with this segment
            if (TRACE) {
                if ((long long)nseg < Q.cap) {
                    if (Q.cells) Q.cells[r * Q.cap + nseg] = cell;
                    if (Q.lens) Q.lens[r * Q.cap + nseg] = len;
                }
                const unsigned cu = (unsigned)cell;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    h ^= (unsigned long long)((cu >> (8 * q)) & 0xffu);
                    h *= 0x100000001b3ULL;
                }
            } else {
                // the record of `cell` was requested one step ago (or at the refill); the next cell's is requested now,
                // before this segment is scored, so that its L2 latency hides behind the score and the next crossing
                const typename Rec::Value cur = rec.value();
                if (!out) rec.load(P.recs, P.ids, P.K, ir_n + nr * iz_n);
                const double S = (double)Rec::sigma(cur, sig, stride, P.K);
                double g, ex;
                score_terms<sizeof(Real) == 8, false>(S, len, g, ex);
                if (len > 0.0) {
                    *st_cell++ = (unsigned)cell;
                    *st_score++ = wa * g;
                    ++k;
                }
                wa *= ex;
            }
            ++nseg;
            t_cur = tn;
            if (out) {
                active = false;
                n_seg += nseg;
                if (TRACE) {
                    if (Q.nseg) Q.nseg[r] = nseg;
                    if (Q.hash) Q.hash[r] = h;
                }
            } else {
                iz = iz_n;
                ir = ir_n;
                if (ax) {                                   // predicated: lanes on a radial step read nothing here
                    pz += stepz;
                    t_z = __dmul_rn(__dsub_rn(lds_f64(ze_addr + 8u * (unsigned)pz), oz), inv_z);
                }
                // One instruction stream for the three kinds of step (axial, inward, outward): the next radial crossing is
                // evaluated every time and kept on a radial step.  It is the inner cylinder of the new shell while the ray still
                // goes inward (ir >= i_turn: D_ir > 0, see the refill), else the outer one: one radius^2 and one discriminant.
                const bool go_in = !ax && inward && ir >= i_turn;
                const double D = rz_disc(bb, a, rho2, lds_f64(re2_addr + 8u * (unsigned)(go_in ? ir : ir + 1)));
                const double sq = __dsqrt_rn(D);
                const double num = go_in ? __dsub_rn(-b, sq) : __dadd_rn(-b, sq);
                const double tq = __dmul_rn(num, inv_a);
                const double tr_new = tq > 0.0 ? tq : 0.0;  // = fmax(0, tq) for every tq (+0 for -0 and for NaN), without the NaN fix-up code
                t_r = ax ? t_r : tr_new;
                inward = ax ? inward : go_in;
            }
        }
        if (!TRACE) {
            __syncwarp();
            const int row = lane % kCoopWindow;
#pragma unroll
            for (int p = 0; p < kCoopWindow; ++p) {
                const int src = p * (32 / kCoopWindow) + lane / kCoopWindow;
                const int kk = __shfl_sync(full, k, src);
                if (row < kk) red_add_f64(P.tally + c_cell[src * (kCoopWindow + 1) + row], c_score[src * (kCoopWindow + 1) + row]);
            }
            __syncwarp();
        }
    }
    if (!TRACE) {
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
}

// ------------------------------------------------------------------------------------------------
// Next-event (point-detector) estimator, SURVEY.md §8(f) NEXT-3 ("requires a ray-cast from
// each source and collision event to the estimator location").  One thread per (event, detector): the same
// S1 look-up and S2/S3 walker, with the UNNORMALISED direction d = det - o so that the crossing parameter
// t = 1 is the detector exactly (steps N1-N6); no tally atomics -- only the optical
// thickness tau = sum_i Sigma_i (l_i R) is carried, and score = W exp(-tau) / R^2 is reduced per CTA into
// the detector's fp64 sum.  blockIdx.y = detector (or P.det_first + blockIdx.y).
//   dynamic shared memory: as cast_kernel.
// ------------------------------------------------------------------------------------------------
struct NextEventParams {
    MeshDev mesh;
    const void *recs;
    const uint8_t *ids;
    int K, M;
    const XsDesc *xs;              // as CastParams
    int N;
    const int *mix_off;
    const int *mix_nuc;
    const void *mix_w;
    const void *rays;
    const uint32_t *perm;          // optional processing order, one section of n entries per detector of the launch
    long long n;
    const double *det;             // [ndet*3] detector points
    int det_first;                 // first detector of this launch
    double *det_sum;               // [ndet] resident sums (may be null in a trace launch)
    unsigned long long *counters;  // [0] accepted pairs [1] rejected pairs [2] segments (may be null)
    // per-event outputs of the test entry point (one detector per launch), any may be null
    uint32_t *nseg;
    unsigned long long *hash;
    double *tau;
    double *score;
};

// accurate exp(-x), x >= 0, from the same reduction as score_terms (full series)
__device__ __forceinline__ double exp_neg(double x)
{
    const double kf = rint(x * -1.4426950408889634074);
    double r = fma(kf, -6.93147180369123816490e-01, -x);
    r = fma(kf, -1.90821492927058770002e-10, r);
    double q = c_expq[0];
#pragma unroll
    for (int i = 1; i < 12; ++i) q = fma(q, r, c_expq[i]);
    const double p = fma(r * r, q, r);
    const int k = (int)kf;
    if (k < -1022) return 0.0;
    const double scale = __longlong_as_double((long long)(k + 1023) << 52);
    return fma(scale, p, scale);
}

template <typename Real, typename Rec, int EDGE_MODE, bool TRACE>
__global__ void __launch_bounds__(256) next_event_kernel(const __grid_constant__ NextEventParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double s_part[8];
    const int stride = blockDim.x;
    unsigned char *sp = smem_raw;
    double *s_edges = reinterpret_cast<double *>(sp);
    if (EDGE_MODE == EDGES_SHARED) sp += edges_smem_bytes_for(P.mesh.nedges);
    AxisF *axf = reinterpret_cast<AxisF *>(sp) + threadIdx.x;
    sp += sizeof(AxisF) * 3 * stride;
    Real *sig = reinterpret_cast<Real *>(sp) + threadIdx.x;
    const double *e = (EDGE_MODE == EDGES_SHARED) ? s_edges : P.mesh.edges;
    if (EDGE_MODE == EDGES_SHARED) {
        for (int i = threadIdx.x; i < P.mesh.nedges; i += blockDim.x) s_edges[i] = __ldg(P.mesh.edges + i);
        __syncthreads();
    }
    const int det = P.det_first + blockIdx.y;
    const double D[3] = {__ldg(P.det + 3 * det), __ldg(P.det + 3 * det + 1), __ldg(P.det + 3 * det + 2)};

    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = i < P.n;
    bool accepted = false;
    unsigned nseg = 0;
    unsigned long long h = 0;
    double tau = 0.0, score = 0.0;
    if (live) {
        const long long r = P.perm ? (long long)__ldg(P.perm + (size_t)blockIdx.y * P.n + i) : i;
        const Ray<Real> R = load_ray<Real>(P.rays, r);
        // N1: only x, y, z, E, W are looked at (the direction fields of the record are ignored)
        const bool fin = isfinite(R.o[0]) && isfinite(R.o[1]) && isfinite(R.o[2]) && isfinite((double)R.E) && isfinite(R.W);
        const double d[3] = {__dsub_rn(D[0], R.o[0]), __dsub_rn(D[1], R.o[1]), __dsub_rn(D[2], R.o[2])};
        const double R2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
        Walker w;
        accepted = fin && (R.E > (Real)0) && isfinite(R2) && (R2 > 0.0) &&
                   walker_init<EDGE_MODE>(w, axf, stride, P.mesh, e, R.o, d);
        if (accepted) {
            const double Rd = sqrt(R2);
            sigma_all<Real>(P.xs, P.M, P.N, P.mix_off, P.mix_nuc, P.mix_w, R.E, sig, stride);   // N2
            if (TRACE) h = 0xcbf29ce484222325ULL;
            Rec rec;
            rec.reset();
            rec.load(P.recs, P.ids, P.K, w.c);
            for (;;) {                                               // N5
                int cell;
                double len;
                const typename Rec::Value cur = rec.value();
                const bool leave = walker_step<EDGE_MODE, true>(w, axf, stride, P.mesh, e, cell, len);
                if (!leave) rec.load(P.recs, P.ids, P.K, w.c);
                const double S = (double)Rec::sigma(cur, sig, stride, P.K);
                tau = fma(S, len * Rd, tau);
                if (TRACE) {
                    const unsigned cu = (unsigned)cell;
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        h ^= (unsigned long long)((cu >> (8 * b)) & 0xffu);
                        h *= 0x100000001b3ULL;
                    }
                }
                ++nseg;
                if (leave) break;
            }
            score = R.W * exp_neg(tau) / R2;                         // N6
        }
        if (TRACE) {
            const long long r = i;                                   // trace launches are never reordered
            if (P.nseg) P.nseg[r] = nseg;
            if (P.hash) P.hash[r] = h;
            if (P.tau) P.tau[r] = tau;
            if (P.score) P.score[r] = score;
        }
    }
    // CTA totals: one fp64 atomic per CTA into the detector's sum, three counter atomics per warp
    const unsigned full = 0xffffffffu;
    double v = score;
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(full, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) s_part[warp] = v;
    const unsigned acc = __popc(__ballot_sync(full, accepted));
    const unsigned rej = __popc(__ballot_sync(full, live && !accepted));
    unsigned long long segs = nseg;
    for (int o = 16; o > 0; o >>= 1) segs += __shfl_xor_sync(full, segs, o);
    if (lane == 0 && P.counters) {
        if (acc) atomicAdd(P.counters + 0, (unsigned long long)acc);
        if (rej) atomicAdd(P.counters + 1, (unsigned long long)rej);
        if (segs) atomicAdd(P.counters + 2, segs);
    }
    __syncthreads();
    if (threadIdx.x == 0 && P.det_sum) {
        double t = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += s_part[i];
        if (t != 0.0) red_add_f64(P.det_sum + det, t);
    }
}

// ------------------------------------------------------------------------------------------------
// Next-event estimator on R-Z and spherical meshes (the NEXT-3 x NEXT-4 cell of SURVEY.md §8(f)):
// steps NZ1-NZ6 of DESIGN.md §10.7 -- the crossing families of rz_kernel (Z4) with the UNNORMALISED direction
// d = det - o, so that t = 1 is the detector; a pending crossing with t >= 1 ends the walk AT the detector; only tau is
// carried; score = W exp(-tau) / R^2.  Work items are (event, detector) pairs, detector-major; persistent lanes as in
// rz_kernel.  A lane keeps the sum of its scores for the detector it is working on and adds it to the detector's
// resident sum when it moves on to the next detector (work items come in detector order), so a launch issues about
// (lanes x detectors) atomics, not one per pair.
//   dynamic shared memory: [edges] [sigma: (M+N) x blockDim Real]
// ------------------------------------------------------------------------------------------------
struct RzNextEventParams {
    CastParams c;                  // mesh (nx = nr, ny = 1), records, tables, rays (events), n; c.counters -> next-event counters
    const double *det;             // [ndet*3] all detector points
    int det_first, ndet;           // detectors of this launch
    double *det_sum;               // resident sums (null in a trace launch)
    unsigned long long *work;      // pair counter, zeroed before the launch
    uint32_t *nseg;                // per-event outputs of the test entry (one detector per launch), any may be null
    unsigned long long *hash;
    double *tau;
    double *score;
    int spherical;
};

template <typename Real, typename Rec, bool TRACE>
__global__ void __launch_bounds__(256) rz_next_event_kernel(const __grid_constant__ RzNextEventParams Q)
{
    const CastParams &P = Q.c;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int stride = blockDim.x;
    const int nr = P.mesh.nx, nz = P.mesh.nz;
    double *s_edges = reinterpret_cast<double *>(smem_raw);
    Real *sig = reinterpret_cast<Real *>(smem_raw + edges_smem_bytes_for(P.mesh.nedges)) + threadIdx.x;
    for (int i = threadIdx.x; i < P.mesh.nedges; i += blockDim.x) s_edges[i] = __ldg(P.mesh.edges + i);
    __syncthreads();
    const double *re = s_edges, *ze = s_edges + nr + 3;
    const bool sph = Q.spherical != 0;
    const unsigned full = 0xffffffffu;
    const unsigned lane = threadIdx.x & 31;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    const long long total = P.n * Q.ndet;

    long long ev = -1;
    bool active = false, inward = false;
    double oz = 0.0, rho2 = 0.0, a = 0.0, b = 0.0, inv_a = 0.0, inv_z = 0.0, t_r = inf, t_z = inf, t_cur = 0.0;
    double W = 0.0, R2 = 1.0, Rd = 0.0, tau = 0.0;
    int ir = 0, iz = 0, pz = 0, stepz = 0;
    unsigned nseg = 0;
    unsigned long long h = 0;
    Rec rec;
    int my_det = -1;                 // detector of the lane's running sum
    double my_sum = 0.0;
    unsigned n_acc = 0, n_rej = 0;
    unsigned long long n_seg = 0;
    bool exhausted = false;

    for (;;) {
        const unsigned idle = __ballot_sync(full, !active);
        if (!exhausted && idle && (__popc(idle) >= kRefillLanes || idle == full)) {
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(Q.work, (unsigned long long)__popc(idle));
            base = __shfl_sync(full, base, 0);
            exhausted = (long long)(base + __popc(idle)) >= total;
            if (!active) {
                const long long q = (long long)base + __popc(idle & ((1u << lane) - 1u));
                if (q < total) {
                    const int j = (int)(q / P.n);
                    ev = q - (long long)j * P.n;
                    const int det = Q.det_first + j;
                    if (det != my_det) {
                        if (!TRACE && my_det >= 0 && my_sum != 0.0) red_add_f64(Q.det_sum + my_det, my_sum);
                        my_det = det;
                        my_sum = 0.0;
                    }
                    double ox, oy;
                    Real E;
                    bool fin;
                    if (sizeof(Real) == 8) {
                        const Ray<double> R = load_ray_f64(P.rays, ev);
                        ox = R.o[0]; oy = R.o[1]; oz = R.o[2]; W = R.W; E = (Real)R.E;
                        fin = isfinite(ox) && isfinite(oy) && isfinite(oz) && isfinite(R.E) && isfinite(W) && R.E > 0.0;
                    } else {
                        const Ray<float> R = load_ray_f32(P.rays, ev);
                        ox = R.o[0]; oy = R.o[1]; oz = R.o[2]; W = R.W; E = (Real)R.E;
                        fin = isfinite(ox) && isfinite(oy) && isfinite(oz) && isfinite((double)R.E) && isfinite(W) && R.E > 0.0f;
                    }
                    // NZ1
                    const double dx = __dsub_rn(__ldg(Q.det + 3 * det), ox), dy = __dsub_rn(__ldg(Q.det + 3 * det + 1), oy),
                                 dz = __dsub_rn(__ldg(Q.det + 3 * det + 2), oz);
                    R2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
                    rho2 = __dadd_rn(__dmul_rn(ox, ox), __dmul_rn(oy, oy));
                    a = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
                    if (sph) {
                        rho2 = __dadd_rn(rho2, __dmul_rn(oz, oz));
                        a = __dadd_rn(a, __dmul_rn(dz, dz));
                    }
                    inv_a = (a != 0.0) ? __drcp_rn(a) : 0.0;
                    const bool radial = (a != 0.0) && isfinite(inv_a) && isfinite(a);
                    inv_z = (dz != 0.0) ? __drcp_rn(dz) : 0.0;
                    const bool axial = !sph && (dz != 0.0) && isfinite(inv_z);
                    const bool accepted = fin && isfinite(R2) && (R2 > 0.0) && (radial || axial) &&
                                          (rho2 < __dmul_rn(re[nr], re[nr])) && (sph || (oz >= ze[0] && oz < ze[nz]));
                    nseg = 0;
                    h = 0;
                    tau = 0.0;
                    if (accepted) {
                        Rd = sqrt(R2);
                        sigma_all<Real>(P.xs, P.M, P.N, P.mix_off, P.mix_nuc, P.mix_w, E, sig, stride);       // NZ2
                        int lo = 0, hi = nr + 1;                                                              // NZ3
                        while (lo < hi) {
                            const int mid = (lo + hi) >> 1;
                            if (__dmul_rn(re[mid], re[mid]) <= rho2) lo = mid + 1; else hi = mid;
                        }
                        ir = lo - 1;
                        iz = sph ? 0 : upper_bound_edges(ze, nz + 1, oz) - 1;
                        b = __dadd_rn(__dmul_rn(ox, dx), __dmul_rn(oy, dy));                                  // NZ4
                        if (sph) b = __dadd_rn(b, __dmul_rn(oz, dz));
                        inward = false;
                        t_r = inf; t_z = inf; t_cur = 0.0; pz = 0; stepz = 0;
                        if (radial) {
                            if (b < 0.0 && ir >= 1) {
                                const double cc = __dsub_rn(rho2, __dmul_rn(re[ir], re[ir]));
                                const double D = __dsub_rn(__dmul_rn(b, b), __dmul_rn(a, cc));
                                if (D > 0.0) { inward = true; t_r = fmax(0.0, __dmul_rn(__dsub_rn(-b, __dsqrt_rn(D)), inv_a)); }
                            }
                            if (!inward) t_r = rz_t_radial(b, a, inv_a, rho2, re[ir + 1], true);
                        }
                        if (axial) {
                            stepz = dz > 0.0 ? 1 : -1;
                            pz = dz > 0.0 ? iz + 1 : iz;
                            t_z = __dmul_rn(__dsub_rn(ze[pz], oz), inv_z);
                        }
                        if (TRACE) h = 0xcbf29ce484222325ULL;
                        rec.reset();
                        active = true;
                        ++n_acc;
                    } else {
                        ++n_rej;
                        if (TRACE) {
                            if (Q.nseg) Q.nseg[ev] = 0;
                            if (Q.hash) Q.hash[ev] = 0;
                            if (Q.tau) Q.tau[ev] = 0.0;
                            if (Q.score) Q.score[ev] = 0.0;
                        }
                    }
                }
            }
        }
        if (__ballot_sync(full, active) == 0) {
            if (exhausted) break;
            continue;
        }
        if (active) {
            // NZ5: one segment
            const bool ax = t_z < t_r;                      // ties: radial first
            const double tn = ax ? t_z : t_r;
            const bool last = tn >= 1.0;                    // the walk ends AT the detector
            const double len = __dsub_rn(last ? 1.0 : tn, t_cur);
            const int cell = ir + nr * iz;
            rec.load(P.recs, P.ids, P.K, cell);
            const double S = (double)Rec::sigma(rec.value(), sig, stride, P.K);
            tau = fma(S, len * Rd, tau);
            if (TRACE) {
                const unsigned cu = (unsigned)cell;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    h ^= (unsigned long long)((cu >> (8 * q)) & 0xffu);
                    h *= 0x100000001b3ULL;
                }
            }
            ++nseg;
            t_cur = tn;
            const int iz_n = ax ? iz + stepz : iz;
            const int ir_n = ax ? ir : (inward ? ir - 1 : ir + 1);
            if (last || iz_n < 0 || iz_n >= nz || ir_n >= nr) {
                active = false;                             // at the detector, or out of the mesh (the rest is void)
                n_seg += nseg;
                const double sc = W * exp_neg(tau) / R2;    // NZ6
                my_sum += sc;
                if (TRACE) {
                    if (Q.nseg) Q.nseg[ev] = nseg;
                    if (Q.hash) Q.hash[ev] = h;
                    if (Q.tau) Q.tau[ev] = tau;
                    if (Q.score) Q.score[ev] = sc;
                }
            } else {
                iz = iz_n;
                ir = ir_n;
                if (ax) {
                    pz += stepz;
                    t_z = __dmul_rn(__dsub_rn(ze[pz], oz), inv_z);
                }
                const bool may_in = !ax && inward && ir >= 1;
                const double rp = re[may_in ? ir : ir + 1];
                const double bb = __dmul_rn(b, b);
                double D = __dsub_rn(bb, __dmul_rn(a, __dsub_rn(rho2, __dmul_rn(rp, rp))));
                bool go_in = may_in && D > 0.0;
                if (may_in && !go_in) {
                    const double ro = re[ir + 1];
                    D = __dsub_rn(bb, __dmul_rn(a, __dsub_rn(rho2, __dmul_rn(ro, ro))));
                }
                const double sq = __dsqrt_rn(D);
                const double num = go_in ? __dsub_rn(-b, sq) : __dadd_rn(-b, sq);
                const double tr_new = fmax(0.0, __dmul_rn(num, inv_a));
                t_r = ax ? t_r : tr_new;
                inward = ax ? inward : go_in;
            }
        }
    }
    if (!TRACE) {
        if (my_det >= 0 && my_sum != 0.0) red_add_f64(Q.det_sum + my_det, my_sum);
        unsigned acc = n_acc, rej = n_rej;
        unsigned long long segs = n_seg;
        for (int o = 16; o > 0; o >>= 1) {
            acc += __shfl_xor_sync(full, acc, o);
            rej += __shfl_xor_sync(full, rej, o);
            segs += __shfl_xor_sync(full, segs, o);
        }
        if (lane == 0 && P.counters) {
            if (acc) atomicAdd(P.counters + 0, (unsigned long long)acc);
            if (rej) atomicAdd(P.counters + 1, (unsigned long long)rej);
            if (segs) atomicAdd(P.counters + 2, segs);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Per-batch moments, SURVEY.md §8(f) NEXT-2 (Eq. (5): FOM = 1/(sigma^2 T), sigma the standard
// deviation of the tally mean).  mr_end_batch folds the batch that just ended:
//     x = tally[c] - prev[c];   s2[c] += x*x;   prev[c] = tally[c]
// (the tally itself stays the running total, so sum_b x_b is the tally).  A pure stream: 40 B per cell.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) fold_batch_kernel(const double *__restrict__ tally, double *__restrict__ prev,
                                                         double *__restrict__ s2, long long ncell)
{
    const long long stride = (long long)gridDim.x * blockDim.x * 2;
    for (long long c = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 2; c < ncell; c += stride) {
        if (c + 1 < ncell) {
            const double2 t = *reinterpret_cast<const double2 *>(tally + c);
            double2 p = *reinterpret_cast<double2 *>(prev + c);
            double2 q = *reinterpret_cast<double2 *>(s2 + c);
            const double x0 = t.x - p.x, x1 = t.y - p.y;
            q.x = fma(x0, x0, q.x);
            q.y = fma(x1, x1, q.y);
            *reinterpret_cast<double2 *>(s2 + c) = q;
            *reinterpret_cast<double2 *>(prev + c) = t;
        } else {
            const double t = tally[c], x = t - prev[c];
            s2[c] = fma(x, x, s2[c]);
            prev[c] = t;
        }
    }
}

// LAYOUT_K4F: move the in-record score sums into the contiguous tally (tally[c] += acc; acc = 0)
__global__ void __launch_bounds__(256) flush_fused_kernel(void *recs, double *__restrict__ tally, long long ncell)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < ncell; c += stride) {
        double *acc = reinterpret_cast<double *>(reinterpret_cast<char *>(recs) + 32 * c + 24);
        const double v = *acc;
        if (v != 0.0) {
            tally[c] += v;
            *acc = 0.0;
        }
    }
}

// mean = prev/B;  sigma = sqrt(max((s2/B - mean^2)/(B-1), 0))   (standard deviation OF THE MEAN; B = 1: +inf)
__global__ void __launch_bounds__(256) mean_sigma_kernel(const double *__restrict__ prev, const double *__restrict__ s2,
                                                         double *__restrict__ mean, double *__restrict__ sigma,
                                                         long long ncell, long long B)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    const double Bd = (double)B;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < ncell; c += stride) {
        const double m = prev[c] / Bd;
        mean[c] = m;
        if (B > 1) {
            const double var = (s2[c] / Bd - m * m) / (double)(B - 1);
            sigma[c] = sqrt(fmax(var, 0.0));
        } else
            sigma[c] = __longlong_as_double(0x7ff0000000000000LL);
    }
}

// ------------------------------------------------------------------------------------------------
// Set-up kernels (mr_load_materials): validate and pack a chunk of the per-cell composition.
//   flags[0] |= 1 on an invalid material id, |= 2 on a non-finite or negative fraction.
// ------------------------------------------------------------------------------------------------
struct PackParams {
    const int32_t *cell_mat;   // chunk, [count*K]
    const double *cell_frac;   // chunk, [count*K]
    const double *density;     // [M]
    long long first, count;    // cells [first, first+count)
    int K, M, layout, is_double;
    void *recs;
    uint8_t *ids;
    int *flags;
};

__global__ void pack_cells_kernel(const PackParams P)
{
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= P.count) return;
    const long long c = P.first + j;
    float rf[MR_PACK_MAX_SLOTS];
    double rd[MR_PACK_MAX_SLOTS];
    unsigned id[MR_PACK_MAX_SLOTS];
    int bad = 0;
    for (int k = 0; k < P.K; ++k) {
        const int m = P.cell_mat[j * P.K + k];
        const double f = P.cell_frac[j * P.K + k];
        if (m < -1 || m >= P.M) { bad |= 1; rd[k] = 0.0; rf[k] = 0.f; id[k] = 0xffu; continue; }
        if (m == -1) { rd[k] = 0.0; rf[k] = 0.f; id[k] = 0xffu; continue; }
        if (!(f >= 0.0) || !isfinite(f)) bad |= 2;
        rd[k] = f * P.density[m];        // r = frac * density, rounded once to fp32 in mixed mode
        rf[k] = (float)rd[k];
        id[k] = (unsigned)m;
    }
    if (bad) atomicOr(P.flags, bad);
    // packed layouts encode an empty slot as r = 0, id = 0 (adds +0 in the same slot order)
    auto pid = [&](int k) { return id[k] == 0xffu ? 0u : id[k]; };
    switch (P.layout) {
    case LAYOUT_K1:
        reinterpret_cast<uint2 *>(P.recs)[c] = make_uint2(__float_as_uint(rf[0]), pid(0));
        break;
    case LAYOUT_K2:
        reinterpret_cast<uint4 *>(P.recs)[c] = make_uint4(__float_as_uint(rf[0]), __float_as_uint(rf[1]), pid(0) | (pid(1) << 8), 0u);
        break;
    case LAYOUT_K3:
        reinterpret_cast<uint4 *>(P.recs)[c] = make_uint4(__float_as_uint(rf[0]), __float_as_uint(rf[1]), __float_as_uint(rf[2]),
                                                         pid(0) | (pid(1) << 8) | (pid(2) << 16));
        break;
    case LAYOUT_K4: {
        uint4 *p = reinterpret_cast<uint4 *>(P.recs) + 2 * c;
        p[0] = make_uint4(__float_as_uint(rf[0]), __float_as_uint(rf[1]), __float_as_uint(rf[2]), __float_as_uint(rf[3]));
        p[1] = make_uint4(pid(0) | (pid(1) << 8) | (pid(2) << 16) | (pid(3) << 24), 0u, 0u, 0u);
        break;
    }
    case LAYOUT_DK3: {
        double *p = reinterpret_cast<double *>(P.recs) + 4 * c;
        p[0] = rd[0];
        p[1] = P.K > 1 ? rd[1] : 0.0;
        p[2] = P.K > 2 ? rd[2] : 0.0;
        reinterpret_cast<uint2 *>(p + 3)[0] = make_uint2(pid(0) | ((P.K > 1 ? pid(1) : 0u) << 8) | ((P.K > 2 ? pid(2) : 0u) << 16), 0u);
        break;
    }
    case LAYOUT_D8: {
        float4 *p = reinterpret_cast<float4 *>(P.recs) + 2 * c;
        p[0] = make_float4(rf[0], rf[1], rf[2], rf[3]);
        p[1] = make_float4(rf[4], rf[5], rf[6], rf[7]);
        break;
    }
    default:
        for (int k = 0; k < P.K; ++k) {
            if (P.is_double) reinterpret_cast<double *>(P.recs)[c * P.K + k] = rd[k];
            else reinterpret_cast<float *>(P.recs)[c * P.K + k] = rf[k];
            P.ids[c * P.K + k] = (uint8_t)id[k];
        }
    }
}

__global__ void convert_f64_to_f32_kernel(const double *in, float *out, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = (float)in[i];
}

}  // namespace mr
