// mr_tiled.cuh -- the cast kernel of the DICTIONARY path (meshes with at most 1024 distinct cell records: configs 1-3),
// S1 -> S6 of DESIGN.md section 1 with the cell bookkeeping done in TILE coordinates (sm_100a).
//
// cast_kernel<TiledRec> (mr_device.cuh) walks in linear cell indices and recomputes (ix, iy, iz) -> (tile, entry) from
// the walker's plane words at every step (17 instructions), and its tally adds go to tally[ix + nx (iy + ny iz)]: lanes
// are unrelated rays, so every add is a request of its own to L2 -- the unit this kernel saturates (lts__t_tag_requests
// 81-87 %, one request per segment; ncu, profiles/).  Here
//   * a ray carries (tag, E): the tile it is in and its (x, y) entry inside the tile, both kept up to date by ONE add
//     per step (E holds the two entry coordinates in separate bit fields with a guard bit each: an entry that leaves the
//     tile clears its guard bit), so the tile id is only recomputed -- incrementally, tag += +-1 | +-ntx | +-ntx nty --
//     when a tile border is crossed;
//   * scores go to TILE-ORDERED accumulators acc[tag * cells_per_tile + entry] (mr_ctx::d_tally_t; moved into the linear
//     tally whenever that is looked at, like the in-record accumulators of section 4.5): consecutive cells of a ray are
//     then neighbours in memory whichever of x and y the ray steps in (a 128-byte line holds 2 rows of 8 cells);
//   * COOP: every lane stages 8 steps' (position, score) pairs in shared memory and the warp adds them TRANSPOSED
//     (MR_OPT_COOP_FLUSH): one instruction carries 8 consecutive segments of each of 4 rays, which now share lines and
//     sectors, so the L2 sees fewer requests than segments;
//   * BITS = 4 (at most 16 distinct records): Sigma_t of every dictionary entry is evaluated once per ray (same fmaf
//     chain in slot order as the per-cell evaluation: bit-identical) into the thread's shared-memory column; a step reads
//     one float;
//   * shared memory is addressed with 32-bit shared-window addresses computed once per thread.
// The crossing parameters, their order (ties x < y < z), the segment lengths and Eq. (4) are those of cast_kernel
// operation by operation (same __dsub_rn / __dmul_rn expressions, same score_terms); only where a score is added changes.
#pragma once
#include "mr_device.cuh"

namespace mr {

template <int BITS> struct TileGeom {
    static constexpr int kXs = BITS == 16 ? 2 : 3;                 // log2 of the tile's x extent
    static constexpr int kYs = BITS == 4 ? 3 : 2;                  // log2 of the tile's y extent
    static constexpr int kCellsLog = kXs + kYs;
    static constexpr unsigned kGuard = (1u << kXs) | (1u << (8 + kYs));
    static constexpr unsigned kWrap = ((1u << kXs) - 1u) | (((1u << kYs) - 1u) << 8);
};

__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void lds_f64x2(unsigned addr, double &a, double &b)
{
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(a), "=d"(b) : "r"(addr));
}
__device__ __forceinline__ float lds_f32(unsigned addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 lds_u32x4(unsigned addr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}

constexpr unsigned kNoPos = 0xffffffffu;      // staged pair that is not to be added (zero-length segment, finished ray)

//   dynamic shared memory: [edges (EDGES_SHARED only)] [walker: 3 x blockDim x 16 B] [sigma: (M+N) x blockDim floats]
//                          [BITS = 4: per-entry Sigma_t: 16 x blockDim floats] [dictionary: ndict x 16 B]
//                          [COOP: per warp 32 x 9 x (8 + 4) bytes]
template <int BITS, int EDGE_MODE, bool COOP>
__global__ void __launch_bounds__(256) cast_tiled_kernel(const __grid_constant__ CastParams P)
{
    using G = TileGeom<BITS>;
    constexpr bool kPerEntry = BITS == 4;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int stride = blockDim.x;
    unsigned char *sp = smem_raw;
    double *s_edges = reinterpret_cast<double *>(sp);
    if (EDGE_MODE == EDGES_SHARED) sp += edges_smem_bytes_for(P.mesh.nedges);
    AxisF *axf = reinterpret_cast<AxisF *>(sp) + threadIdx.x;
    sp += sizeof(AxisF) * 3 * stride;
    float *sig = reinterpret_cast<float *>(sp) + threadIdx.x;
    sp += (sizeof(float) * (size_t)(P.M + P.N) * stride + 15) & ~(size_t)15;
    float *sig_e = reinterpret_cast<float *>(sp) + threadIdx.x;
    if (kPerEntry) sp += sizeof(float) * (size_t)kPerEntryMax * stride;
    uint4 *s_dict = reinterpret_cast<uint4 *>(sp);
    sp += sizeof(uint4) * (size_t)P.ndict;
    double *c_score = reinterpret_cast<double *>(sp + (threadIdx.x >> 5) * coop_warp_smem_bytes());
    unsigned *c_pos = reinterpret_cast<unsigned *>(c_score + 32 * (kCoopWindow + 1));
    const double *e = (EDGE_MODE == EDGES_SHARED) ? s_edges : P.mesh.edges;
    if (EDGE_MODE == EDGES_SHARED) {
        for (int i = threadIdx.x; i < P.mesh.nedges; i += blockDim.x) s_edges[i] = __ldg(P.mesh.edges + i);
    }
    for (int i = threadIdx.x; i < P.ndict; i += blockDim.x) s_dict[i] = __ldg(P.dict + i);
    __syncthreads();
    const unsigned axf_addr = smem_addr(axf), axf_step = (unsigned)stride * (unsigned)sizeof(AxisF);
    const unsigned sige_addr = smem_addr(sig_e), sig_step = (unsigned)stride * 4u;
    const unsigned dict_addr = smem_addr(s_dict);

    const unsigned full = 0xffffffffu;
    const unsigned lane = threadIdx.x & 31;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = i < P.n;
    bool accepted = false;
    unsigned nseg = 0;

    // walker state (registers): pending crossing parameters, packed plane words, step signs; tile id, entry word, tile
    double t0 = 0.0, t1 = 0.0, t2 = 0.0, tcur = 0.0, wa = 0.0;
    int pl0 = 0, pl1 = 0, pl2 = 0, s0 = 0, s1 = 0, s2 = 0;
    int tag = 0;
    unsigned E = 0;
    uint4 ta = make_uint4(0, 0, 0, 0), tb = make_uint4(0, 0, 0, 0);
    const int ntx = P.ntx, ntxy = P.ntx * P.nty;
    double *const acc = P.tally_t;

    if (live) {
        const long long r = P.perm ? (long long)__ldg(P.perm + i) : i;
        const Ray<float> R = load_ray<float>(P.rays, r);
        Walker w;
        accepted = R.finite && (R.E > 0.f) && walker_init<EDGE_MODE>(w, axf, stride, P.mesh, e, R.o, R.d);
        if (accepted) {
            sigma_all<float>(P.xs, P.M, P.N, P.mix_off, P.mix_nuc, P.mix_w, R.E, sig, stride);
            if (kPerEntry)
                for (int q = 0; q < P.ndict; ++q) sig_e[q * stride] = TiledRec<BITS>::sigma_rec(s_dict[q], sig, stride, P.K);
            wa = R.W;
            t0 = w.t0; t1 = w.t1; t2 = w.t2;
            pl0 = w.pl0; pl1 = w.pl1; pl2 = w.pl2;
            s0 = (w.dc0 > 0) - (w.dc0 < 0); s1 = (w.dc1 > 0) - (w.dc1 < 0); s2 = (w.dc2 > 0) - (w.dc2 < 0);
            const int ix = walker_cell_index(w.pl0, w.dc0), iy = walker_cell_index(w.pl1, w.dc1), iz = walker_cell_index(w.pl2, w.dc2);
            tag = (ix >> G::kXs) + ntx * (iy >> G::kYs) + ntxy * iz;
            E = (((unsigned)ix & ((1u << G::kXs) - 1u)) | (((unsigned)iy & ((1u << G::kYs) - 1u)) << 8)) | G::kGuard;
            ldg_256(P.tiles + 2 * (size_t)tag, ta, tb);
        }
    }
    __syncwarp();                                                      // the shared-memory columns are read through asm below
    bool left = !accepted;

    // One segment (O5): returns true if the segment has positive length (a zero-length one scores exactly 0);
    // pos = where its score goes in the tile-ordered accumulators, v = the score; `left` is set when the ray is out.
    auto segment = [&](unsigned &pos, double &v) {
        const bool ysel = t1 < t0;                     // ties keep x
        const double tm = ysel ? t1 : t0;
        const bool zsel = t2 < tm;                     // ties keep x / y
        const double tn = zsel ? t2 : tm;
        const int a = zsel ? 2 : (ysel ? 1 : 0);
        const int pl = zsel ? pl2 : (ysel ? pl1 : pl0);
        const int s = zsel ? s2 : (ysel ? s1 : s0);
        double ao, aiv;
        lds_f64x2(axf_addr + (unsigned)a * axf_step, ao, aiv);
        const double len = __dsub_rn(tn, tcur);
        tcur = tn;
        // the cell just traversed: entry in the resident tile -> Sigma_t, position in the accumulators
        const unsigned en = (((E >> 8) << G::kXs) | (E & ((1u << G::kXs) - 1u))) & ((1u << G::kCellsLog) - 1u);
        pos = ((unsigned)tag << G::kCellsLog) | en;
        const unsigned bit = en * BITS;
        const unsigned rr = bit >> 5;
        const uint32_t lo4 = (rr & 2) ? ((rr & 1) ? ta.w : ta.z) : ((rr & 1) ? ta.y : ta.x);
        const uint32_t hi4 = (rr & 2) ? ((rr & 1) ? tb.w : tb.z) : ((rr & 1) ? tb.y : tb.x);
        const unsigned idx = (((rr & 4) ? hi4 : lo4) >> (bit & 31)) & ((1u << BITS) - 1u);
        float Sf;
        if (kPerEntry) Sf = lds_f32(sige_addr + idx * sig_step);
        else Sf = TiledRec<BITS>::sigma_rec(lds_u32x4(dict_addr + idx * 16u), sig, stride, P.K);
        // the walker's update (O4), as walker_step
        const int p = pl & 0xffff;
        const bool leave = (p == (int)((unsigned)pl >> 16));
        const int adv = leave ? 0 : s;
        const int pq = p + adv;                        // never read outside the table
        const int base = (EDGE_MODE == EDGES_ARITH) ? 0 : (zsel ? P.mesh.nx + P.mesh.ny + 2 : (ysel ? P.mesh.nx + 1 : 0));
        const double tnew = __dmul_rn(__dsub_rn(plane_pos<EDGE_MODE>(P.mesh, e, a, base, pq), ao), aiv);
        const int pln = pl + adv;                      // a ray that is out stays where it is: stepping it again "leaves" again
        t0 = (zsel || ysel) ? t0 : tnew;
        t1 = (!zsel && ysel) ? tnew : t1;
        t2 = zsel ? tnew : t2;
        pl0 = (zsel || ysel) ? pl0 : pln;
        pl1 = (!zsel && ysel) ? pln : pl1;
        pl2 = zsel ? pln : pl2;
        // the next cell: one add moves the entry; a cleared guard bit (or any z step) means another tile
        E += (unsigned)s << (8 * a);
        if (!leave && (zsel || (~E & G::kGuard) != 0u)) {
            tag += s * (zsel ? ntxy : (ysel ? ntx : 1));
            E = (E & G::kWrap) | G::kGuard;
            ldg_256(P.tiles + 2 * (size_t)tag, ta, tb);
        }
        // S5
        double g, ex;
        score_terms<false>((double)Sf, len, g, ex);
        v = wa * g;
        wa *= ex;
        ++nseg;
        left = leave;
        return len > 0.0;
    };

    // the first P.agg_first segments of a ray with warp-aggregated atomics (rays born in one small region, section 4.7)
    for (int k = 0; k < P.agg_first; ++k) {
        if (!left) {
            unsigned pos;
            double v;
            bool add = segment(pos, v);
            const unsigned act = __activemask();
            const unsigned peers = __match_any_sync(act, add ? pos : 0x80000000u | lane);
            if (peers & (peers - 1)) {
                const int leader = __ffs(peers) - 1;
                double sum = 0.0;
                for (unsigned rest = peers; rest; rest &= rest - 1) sum += __shfl_sync(peers, v, __ffs(rest) - 1);
                v = sum;
                add = add && (int)lane == leader;
            }
            if (add) red_add_f64(acc + pos, v);
        }
    }
    if (COOP) {
        // windows of kCoopWindow steps staged per lane, then the transposed adds
        while (__any_sync(full, !left)) {
#pragma unroll 1
            for (int j = 0; j < kCoopWindow; ++j) {
                // no branch around the step: a lane whose ray is out keeps stepping in place (its plane word says "leave"
                // again, it loads nothing) and its pair is flagged kNoPos
                const bool was_left = left;
                double v;
                unsigned q;
                const bool pos_len = segment(q, v);
                c_score[lane * (kCoopWindow + 1) + j] = v;
                c_pos[lane * (kCoopWindow + 1) + j] = (pos_len && !was_left) ? q : kNoPos;
                nseg -= was_left ? 1u : 0u;
                left = left || was_left;
            }
            __syncwarp();
            const int row = lane % kCoopWindow;
#pragma unroll
            for (int p = 0; p < kCoopWindow; ++p) {
                const int src = p * (32 / kCoopWindow) + lane / kCoopWindow;
                const unsigned pos = c_pos[src * (kCoopWindow + 1) + row];
                if (pos != kNoPos) red_add_f64(acc + pos, c_score[src * (kCoopWindow + 1) + row]);
            }
            __syncwarp();
        }
    } else {
        while (!left) {
            unsigned pos;
            double v;
            if (segment(pos, v)) red_add_f64(acc + pos, v);
        }
    }
    const unsigned nacc = __popc(__ballot_sync(full, accepted));
    const unsigned nrej = __popc(__ballot_sync(full, live && !accepted));
    unsigned long long segs = nseg;
    for (int o = 16; o > 0; o >>= 1) segs += __shfl_xor_sync(full, segs, o);
    if (lane == 0) {
        if (nacc) atomicAdd(P.counters + 0, (unsigned long long)nacc);
        if (nrej) atomicAdd(P.counters + 1, (unsigned long long)nrej);
        if (segs) atomicAdd(P.counters + 2, segs);
    }
}

// ------------------------------------------------------------------------------------------------
// Next-event cast (NEXT-3, steps N1-N6 of DESIGN.md section 10.3) on the dictionary path with at most 16 distinct records:
// next_event_kernel with the walk in tile coordinates -- tile id and entry word as in cast_tiled_kernel, Sigma_t of every
// dictionary entry evaluated once per (event, detector) pair -- so that a step costs one 4-byte shared load and, every
// fifth step or so, one 32-byte index tile, where the record-pair path costs 0.65 uncoalesced record loads and K sigma
// reads per step (that kernel sits on the LSU pipe, 82 %, and on instruction issue, 80 %).  Crossing parameters, their
// order, the end at t = 1 and tau are those of next_event_kernel operation by operation; the linear cell index (needed for
// the FNV hash of the test entry only) is rebuilt from (tile, entry).
//   dynamic shared memory: [edges (EDGES_SHARED only)] [walker: 3 x blockDim x 16 B] [sigma: (M+N) x blockDim floats]
//                          [per-entry Sigma_t: 16 x blockDim floats] [dictionary: ndict x 16 B]
// ------------------------------------------------------------------------------------------------
struct NextEventTiles {
    const uint4 *dict;
    const uint4 *tiles;
    int ndict, ntx, nty;
};

template <int EDGE_MODE, bool TRACE>
__global__ void __launch_bounds__(256) next_event_tiled_kernel(const __grid_constant__ NextEventParams P, const __grid_constant__ NextEventTiles T)
{
    using G = TileGeom<4>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double s_part[8];
    const int stride = blockDim.x;
    unsigned char *sp = smem_raw;
    double *s_edges = reinterpret_cast<double *>(sp);
    if (EDGE_MODE == EDGES_SHARED) sp += edges_smem_bytes_for(P.mesh.nedges);
    AxisF *axf = reinterpret_cast<AxisF *>(sp) + threadIdx.x;
    sp += sizeof(AxisF) * 3 * stride;
    float *sig = reinterpret_cast<float *>(sp) + threadIdx.x;
    sp += (sizeof(float) * (size_t)(P.M + P.N) * stride + 15) & ~(size_t)15;
    float *sig_e = reinterpret_cast<float *>(sp) + threadIdx.x;
    sp += sizeof(float) * (size_t)kPerEntryMax * stride;
    uint4 *s_dict = reinterpret_cast<uint4 *>(sp);
    const double *e = (EDGE_MODE == EDGES_SHARED) ? s_edges : P.mesh.edges;
    if (EDGE_MODE == EDGES_SHARED) {
        for (int i = threadIdx.x; i < P.mesh.nedges; i += blockDim.x) s_edges[i] = __ldg(P.mesh.edges + i);
    }
    for (int i = threadIdx.x; i < T.ndict; i += blockDim.x) s_dict[i] = __ldg(T.dict + i);
    __syncthreads();
    const unsigned axf_addr = smem_addr(axf), axf_step = (unsigned)stride * (unsigned)sizeof(AxisF);
    const unsigned sige_addr = smem_addr(sig_e), sig_step = (unsigned)stride * 4u;
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
        const Ray<float> R = load_ray<float>(P.rays, r);
        // N1: only x, y, z, E, W are looked at (the direction fields of the record are ignored)
        const bool fin = isfinite(R.o[0]) && isfinite(R.o[1]) && isfinite(R.o[2]) && isfinite((double)R.E) && isfinite(R.W);
        const double d[3] = {__dsub_rn(D[0], R.o[0]), __dsub_rn(D[1], R.o[1]), __dsub_rn(D[2], R.o[2])};
        const double R2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
        Walker w;
        accepted = fin && (R.E > 0.f) && isfinite(R2) && (R2 > 0.0) && walker_init<EDGE_MODE>(w, axf, stride, P.mesh, e, R.o, d);
        if (accepted) {
            const double Rd = sqrt(R2);
            sigma_all<float>(P.xs, P.M, P.N, P.mix_off, P.mix_nuc, P.mix_w, R.E, sig, stride);   // N2
            for (int q = 0; q < T.ndict; ++q) sig_e[q * stride] = TiledRec<4>::sigma_rec(s_dict[q], sig, stride, P.K);
            asm volatile("" ::: "memory");                          // the column is read through asm loads below: keep the stores above them
            if (TRACE) h = 0xcbf29ce484222325ULL;
            double t0 = w.t0, t1 = w.t1, t2 = w.t2, tcur = 0.0;
            int pl0 = w.pl0, pl1 = w.pl1, pl2 = w.pl2;
            const int s0 = (w.dc0 > 0) - (w.dc0 < 0), s1 = (w.dc1 > 0) - (w.dc1 < 0), s2 = (w.dc2 > 0) - (w.dc2 < 0);
            const int ix = walker_cell_index(w.pl0, w.dc0), iy = walker_cell_index(w.pl1, w.dc1), iz = walker_cell_index(w.pl2, w.dc2);
            const int ntx = T.ntx, ntxy = T.ntx * T.nty;
            int tag = (ix >> G::kXs) + ntx * (iy >> G::kYs) + ntxy * iz;
            unsigned E = (((unsigned)ix & ((1u << G::kXs) - 1u)) | (((unsigned)iy & ((1u << G::kYs) - 1u)) << 8)) | G::kGuard;
            uint4 ta, tb;
            ldg_256(T.tiles + 2 * (size_t)tag, ta, tb);
            for (;;) {                                               // N5
                const bool ysel = t1 < t0;                           // ties keep x
                const double tm = ysel ? t1 : t0;
                const bool zsel = t2 < tm;                           // ties keep x / y
                const double tn = zsel ? t2 : tm;
                // the cell the walker stands in: entry of the resident tile -> Sigma_t
                const unsigned en = (((E >> 8) << G::kXs) | (E & ((1u << G::kXs) - 1u))) & ((1u << G::kCellsLog) - 1u);
                const unsigned bit = en * 4u;
                const unsigned rr = bit >> 5;
                const uint32_t lo4 = (rr & 2) ? ((rr & 1) ? ta.w : ta.z) : ((rr & 1) ? ta.y : ta.x);
                const uint32_t hi4 = (rr & 2) ? ((rr & 1) ? tb.w : tb.z) : ((rr & 1) ? tb.y : tb.x);
                const unsigned idx = (((rr & 4) ? hi4 : lo4) >> (bit & 31)) & 15u;
                const float Sf = lds_f32(sige_addr + idx * sig_step);
                if (TRACE) {
                    // linear cell index from (tile, entry): tile = tx + ntx * (ty + nty * iz)
                    const int tz = tag / ntxy, trem = tag - tz * ntxy, ty = trem / ntx, tx = trem - ty * ntx;
                    const unsigned cu = (unsigned)(((tx << G::kXs) | (int)(en & ((1u << G::kXs) - 1u))) +
                                                   P.mesh.nx * (((ty << G::kYs) | (int)(en >> G::kXs)) + P.mesh.ny * tz));
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        h ^= (unsigned long long)((cu >> (8 * b)) & 0xffu);
                        h *= 0x100000001b3ULL;
                    }
                }
                ++nseg;
                if (tn >= 1.0) {                                     // the pending crossing lies beyond the detector: the walk ends AT it
                    tau = fma((double)Sf, __dsub_rn(1.0, tcur) * Rd, tau);
                    break;
                }
                const int a = zsel ? 2 : (ysel ? 1 : 0);
                const int pl = zsel ? pl2 : (ysel ? pl1 : pl0);
                const int s = zsel ? s2 : (ysel ? s1 : s0);
                double ao, aiv;
                lds_f64x2(axf_addr + (unsigned)a * axf_step, ao, aiv);
                const double len = __dsub_rn(tn, tcur);
                tcur = tn;
                tau = fma((double)Sf, len * Rd, tau);
                const int p = pl & 0xffff;
                if (p == (int)((unsigned)pl >> 16)) break;           // left the mesh (outside is void)
                const int pq = p + s;
                const int base = (EDGE_MODE == EDGES_ARITH) ? 0 : (zsel ? P.mesh.nx + P.mesh.ny + 2 : (ysel ? P.mesh.nx + 1 : 0));
                const double tnew = __dmul_rn(__dsub_rn(plane_pos<EDGE_MODE>(P.mesh, e, a, base, pq), ao), aiv);
                const int pln = pl + s;
                t0 = (zsel || ysel) ? t0 : tnew;
                t1 = (!zsel && ysel) ? tnew : t1;
                t2 = zsel ? tnew : t2;
                pl0 = (zsel || ysel) ? pl0 : pln;
                pl1 = (!zsel && ysel) ? pln : pl1;
                pl2 = zsel ? pln : pl2;
                E += (unsigned)s << (8 * a);
                if (zsel || (~E & G::kGuard) != 0u) {
                    tag += s * (zsel ? ntxy : (ysel ? ntx : 1));
                    E = (E & G::kWrap) | G::kGuard;
                    ldg_256(T.tiles + 2 * (size_t)tag, ta, tb);
                }
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

// Moves the tile-ordered accumulators into the linear tally (tally[c] += acc[pos(c)]; acc = 0).  One thread per cell of
// the linear order; xs / ys = log2 of the tile extents.
__global__ void __launch_bounds__(256) flush_tiled_kernel(double *__restrict__ acc, double *__restrict__ tally, int nx, int ny, int nz,
                                                          int ntx, int nty, int xs, int ys)
{
    const long long ncell = (long long)nx * ny * nz;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < ncell; c += stride) {
        const int ix = (int)(c % nx), iy = (int)((c / nx) % ny), iz = (int)(c / ((long long)nx * ny));
        const long long tag = (ix >> xs) + (long long)ntx * ((iy >> ys) + (long long)nty * iz);
        const long long pos = (tag << (xs + ys)) | (((iy & ((1 << ys) - 1)) << xs) | (ix & ((1 << xs) - 1)));
        const double v = acc[pos];
        if (v != 0.0) {
            tally[c] += v;
            acc[pos] = 0.0;
        }
    }
}

}  // namespace mr
