// mr_persist.cuh -- the cast kernel with PERSISTENT lanes (sm_100a): S1 -> S6 as cast_kernel / cast_coop_kernel, but a lane
// whose ray has left the mesh takes the next ray from a global counter instead of idling until the longest ray of its
// CTA is done.
//
// cast_kernel gives every thread one ray: a CTA lives as long as its longest ray, the grid ends in a tail of half-empty
// SMs, and every launch ramps up and down for about 0.2 ms.  On the 10^7-ray batch that is 3 % of the kernel; on a
// 10^6-ray batch (config 2) and on the 2^18 .. 2^21-ray chunks a HOST batch is cast in (mr_cast_rays from host memory, the
// producer ring) it is 15-25 %.  Here the grid is as many CTAs as are resident at once, rays are handed out in the order
// of the ordering pre-pass (so its z-slab locality and its longest-first order survive: lanes that refill together
// take consecutive rays), and refills are batched (at least kPersistRefill idle lanes of a warp, or nothing left to
// wait for), because the per-ray set-up (S1, S2) is divergent code.
//   COOP: the transposed tally adds of cast_coop_kernel (8 steps staged per lane, then 8 consecutive segments of 4 rays per
//         instruction); else one RED per segment straight from the walking lane.
//   The first P.agg_first segments of a ray are warp-aggregated as in cast_kernel (section 4.7), among the lanes that are
//   in their first segments at the same step (lanes that were refilled together).
// Scores, cells and their order per ray are those of cast_kernel; tally[c] receives the same values in another order (Q18).
//   dynamic shared memory: as cast_coop_kernel ([edges] [walker] [sigma] [per-entry sigma] [dictionary] [per warp staging]).
#pragma once
#include "mr_device.cuh"

namespace mr {

constexpr int kPersistRefill = 8;
constexpr int kPersistWindow = kCoopWindow;   // steps between two looks at the idle lanes

template <typename Real, typename Rec, int EDGE_MODE, bool COOP>
__global__ void __launch_bounds__(256) cast_persist_kernel(const __grid_constant__ CastParams P, unsigned long long *__restrict__ work)
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
    bool active = false, exhausted = false;
    unsigned nseg = 0;                       // segments of the lane's current ray
    unsigned n_acc = 0, n_rej = 0;
    unsigned long long n_seg = 0;
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
    for (;;) {
        // ---- refill the idle lanes (batched)
        const unsigned idle = __ballot_sync(full, !active);
        if (!exhausted && idle && (__popc(idle) >= kPersistRefill || idle == full)) {
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(work, (unsigned long long)__popc(idle));
            base = __shfl_sync(full, base, 0);
            exhausted = (long long)(base + __popc(idle)) >= P.n;
            if (!active) {
                const long long i = (long long)base + __popc(idle & ((1u << lane) - 1u));
                if (i < P.n) {
                    const long long r = P.perm ? (long long)__ldg(P.perm + i) : i;
                    const Ray<Real> R = load_ray<Real>(P.rays, r);
                    const bool accepted = R.finite && (R.E > (Real)0) && walker_init<EDGE_MODE>(w, axf, stride, P.mesh, e, R.o, R.d);
                    if (accepted) {
                        sigma_all<Real>(P.xs, P.M, P.N, P.mix_off, P.mix_nuc, P.mix_w, R.E, sig, stride);
                        if constexpr (kPerEntry)
                            for (int q = 0; q < P.ndict; ++q) sig_e[q * stride] = Rec::sigma_rec(s_dict[q], sig, stride, P.K);
                        wa = R.W;
                        nseg = 0;
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
        // ---- kPersistWindow steps
        int k = 0;
#pragma unroll 1
        for (int j = 0; j < kPersistWindow; ++j) {
            if (active) {
                int cell;
                double len;
                const bool leave = walker_step<EDGE_MODE>(w, axf, stride, P.mesh, e, cell, len);
                typename Rec::Value cur;
                if constexpr (Rec::kTiled) cur = rec.value(s_dict, (const float *)sig_e, stride);
                else cur = rec.value();
                if (!leave) fetch();
                const double S = (double)Rec::sigma(cur, sig, stride, P.K);
                double g, ex;
                score_terms<sizeof(Real) == 8>(S, len, g, ex);
                double v = wa * g;
                wa *= ex;
                bool add = len > 0.0;
                // the first P.agg_first segments of a ray: lanes of the warp that score into the same cell add once
                const unsigned young = __ballot_sync(__activemask(), nseg < (unsigned)P.agg_first);
                if (young) {
                    const bool mine = nseg < (unsigned)P.agg_first;
                    const unsigned peers = __match_any_sync(__activemask(), (add && mine) ? cell : -1 - (int)lane);
                    if (peers & (peers - 1)) {
                        const int leader = __ffs(peers) - 1;
                        double sum = 0.0;
                        for (unsigned rest = peers; rest; rest &= rest - 1) sum += __shfl_sync(peers, v, __ffs(rest) - 1);
                        v = sum;
                        add = add && (int)lane == leader;
                    }
                }
                ++nseg;
                if (add) {
                    if (COOP) {
                        c_cell[lane * (kCoopWindow + 1) + k] = (unsigned)cell;
                        c_score[lane * (kCoopWindow + 1) + k] = v;
                        ++k;
                    } else
                        red_add_f64(Rec::tally_at(P.tally, P.recs, cell), v);
                }
                if (leave) {
                    active = false;
                    n_seg += nseg;
                }
            }
        }
        if (COOP) {
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

}  // namespace mr
