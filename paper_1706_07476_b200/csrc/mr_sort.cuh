// mr_sort.cuh -- batch pre-pass: order the rays of a batch by (start z-slab, estimated segment count).
//
// Why (DESIGN.md §4 "ray ordering"): one thread walks one ray, so a warp runs as long as its longest
// ray and touches cell records / tally lines wherever its 32 rays happen to be.  Ordering a batch so
// that (a) rays of one warp need about the same number of steps and (b) CTAs resident at the same
// time work in the same few z-slabs raises lane utilisation and keeps the working set (a z-slab of
// records + tally is contiguous in memory, x fastest) inside the 126 MB L2.  The order only changes
// which thread walks which ray: every ray's trace and score are unchanged, and the tally differs by
// fp64 summation order only (reading Q18).
//
// Three kernels: classify (key per ray + histogram), scan (exclusive prefix over the keys), scatter
// (ray index -> sorted position).  A counting sort: O(n), no library call.
#pragma once
#include "mr_device.cuh"

namespace mr {

struct SortParams {
    MeshDev mesh;
    const void *rays;
    long long n;
    int ray_is_double;
    int zdiv;        // z-slab thickness in cells
    int lshift;      // estimated segments >> lshift = length bucket
    int nlen;        // length buckets per slab
    int nkeys;       // slabs * nlen + 1 (last key: rejected rays)
    uint32_t *keys;  // [n]
    uint32_t *hist;  // [nkeys + 1], zeroed before classify; becomes the exclusive prefix after scan
    uint32_t *perm;  // [n]
    // next-event mode (det != null): blockIdx.y = detector det_first + y; the "direction" of ray r is det - origin,
    // the walk ends at the detector (t = 1); keys / hist / perm hold one section per detector of the launch
    const double *det;
    int det_first;
    // 1: length-major order, longest rays first (working set fits in L2, so slab locality buys nothing and the
    // kernel's tail -- the last CTAs still walking long rays -- is what costs); 0: slab-major, length within a slab
    int longest_first;
    int nslab;
    int arith;       // the mesh is arithmetic (MeshDev::e0, h valid): cell indices by one multiply instead of a search
    // block-local variant (count_kernel ... place_kernel): CTA b of a section owns rays [n*b/nblk, n*(b+1)/nblk)
    int nblk;
    uint32_t *blk_hist;   // [sections][nblk][nkeys]: per-CTA counts, then per-CTA first output positions
};

// key of ray r for the section (detector) of this CTA; e = the plane table staged in shared memory
__device__ __forceinline__ uint32_t ray_key(const SortParams &P, const double *e, long long r)
{
    // the key only orders the work: an index that is off by one near a plane is harmless here
    auto cell_of = [&](int a, int base, int n, double x) {
        if (P.arith) return min(max((int)floor((x - P.mesh.e0[a]) / P.mesh.h[a]), 0), n - 1);
        return min(max(upper_bound_edges(e + base, n + 1, x) - 1, 0), n - 1);
    };
    double o[3], d[3];
    bool ok;
    if (P.ray_is_double) {
        const Ray<double> R = load_ray_f64(P.rays, r);
        for (int a = 0; a < 3; ++a) { o[a] = R.o[a]; d[a] = R.d[a]; }
        ok = (P.det ? (isfinite(o[0]) && isfinite(o[1]) && isfinite(o[2]) && isfinite(R.E) && isfinite(R.W)) : R.finite) && R.E > 0.0;
    } else {
        const Ray<float> R = load_ray_f32(P.rays, r);
        for (int a = 0; a < 3; ++a) { o[a] = R.o[a]; d[a] = R.d[a]; }
        ok = (P.det ? (isfinite(o[0]) && isfinite(o[1]) && isfinite(o[2]) && isfinite(R.E) && isfinite(R.W)) : R.finite) && R.E > 0.0f;
    }
    if (P.det) {
        const double *D = P.det + 3 * (size_t)(P.det_first + blockIdx.y);
        for (int a = 0; a < 3; ++a) d[a] = __ldg(D + a) - o[a];
        ok = ok && isfinite(d[0]) && isfinite(d[1]) && isfinite(d[2]);
    }
    const int base[3] = {0, P.mesh.nx + 1, P.mesh.nx + P.mesh.ny + 2};
    const int n[3] = {P.mesh.nx, P.mesh.ny, P.mesh.nz};
    int idx[3] = {0, 0, 0};
    if (P.arith) {
        // arithmetic mesh: the whole estimate in fp32 -- nine fp64 divisions per ray made this pass fp64-pipe bound
        // (64 lanes per clock per SM).  The key only orders the work: an index that is off by one near a plane, or a
        // ray on the box surface that lands in the last bucket, is harmless.
        uint32_t key = (uint32_t)(P.nkeys - 1);
        float of[3], df[3], ih[3], span[3], t_exit = __int_as_float(0x7f800000);
        for (int a = 0; a < 3 && ok; ++a) {
            of[a] = (float)(o[a] - P.mesh.e0[a]);
            df[a] = (float)d[a];
            ih[a] = __frcp_rn((float)P.mesh.h[a]);
            span[a] = (float)n[a] * (float)P.mesh.h[a];
            ok = of[a] >= 0.f && of[a] < span[a];
            idx[a] = min((int)(of[a] * ih[a]), n[a] - 1);
            if (df[a] != 0.f) t_exit = fminf(t_exit, __fdividef((df[a] > 0.f ? span[a] : 0.f) - of[a], df[a]));
        }
        if (P.det) t_exit = fminf(t_exit, 1.0f);   // the walk ends at the detector
        if (ok && isfinite(t_exit)) {
            int est = 1;   // cells crossed ~ 1 + sum of index distances between the origin and the exit point
            for (int a = 0; a < 3; ++a) {
                const float x = fminf(fmaxf(fmaf(t_exit, df[a], of[a]), 0.f), span[a]);
                est += abs(min((int)(x * ih[a]), n[a] - 1) - idx[a]);
            }
            const int lb = min(est >> P.lshift, P.nlen - 1);
            key = P.longest_first ? (uint32_t)((P.nlen - 1 - lb) * P.nslab + idx[2] / P.zdiv)
                                  : (uint32_t)((idx[2] / P.zdiv) * P.nlen + lb);
        }
        return key;
    }
    double t_exit = __longlong_as_double(0x7ff0000000000000LL);
    for (int a = 0; a < 3 && ok; ++a) {
        ok = (o[a] >= e[base[a]] && o[a] < e[base[a] + n[a]]);
        if (!ok) break;
        idx[a] = cell_of(a, base[a], n[a], o[a]);
        if (d[a] != 0.0) {
            const double t = (e[base[a] + (d[a] > 0.0 ? n[a] : 0)] - o[a]) / d[a];
            t_exit = fmin(t_exit, t);
        }
    }
    if (P.det) t_exit = fmin(t_exit, 1.0);   // the walk ends at the detector
    ok = ok && isfinite(t_exit);
    uint32_t key = (uint32_t)(P.nkeys - 1);
    if (ok) {
        int est = 1;   // cells crossed ~ 1 + sum of index distances between the origin and the exit point
        for (int a = 0; a < 3; ++a) {
            double x = fma(t_exit, d[a], o[a]);
            x = fmin(fmax(x, e[base[a]]), e[base[a] + n[a]]);
            est += abs(cell_of(a, base[a], n[a], x) - idx[a]);
        }
        const int lb = min(est >> P.lshift, P.nlen - 1);
        key = P.longest_first ? (uint32_t)((P.nlen - 1 - lb) * P.nslab + idx[2] / P.zdiv)
                              : (uint32_t)((idx[2] / P.zdiv) * P.nlen + lb);
    }
    return key;
}

// dynamic shared memory: [edges] (always staged: the search would otherwise hammer global memory)
__global__ void __launch_bounds__(256) classify_kernel(const SortParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *e = reinterpret_cast<double *>(smem_raw);
    for (int i = threadIdx.x; i < P.mesh.nedges; i += blockDim.x) e[i] = __ldg(P.mesh.edges + i);
    __syncthreads();
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= P.n) return;
    const uint32_t key = ray_key(P, e, r);
    const size_t sec = P.det ? blockIdx.y : 0;
    P.keys[sec * P.n + r] = key;
    // one atomic per distinct key of the warp (rays born in one small region share a handful of keys)
    const unsigned act = __activemask();
    const unsigned peers = __match_any_sync(act, key);
    if ((int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(P.hist + sec * (P.nkeys + 1) + key, (unsigned)__popc(peers));
}

// ---- block-local counting sort (no global atomics: 10^7 random global atomics cost ~0.22 ms in each of classify and
//      scatter; shared-memory counters cost a fifth of that).  grid = (nblk, sections), 1024 threads.
//      dynamic shared memory: [edges] [counters: nkeys u32]
__global__ void __launch_bounds__(1024) count_kernel(const SortParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *e = reinterpret_cast<double *>(smem_raw);
    uint32_t *cnt = reinterpret_cast<uint32_t *>(smem_raw + sizeof(double) * (size_t)((P.mesh.nedges + 1) & ~1));
    for (int i = threadIdx.x; i < P.mesh.nedges; i += blockDim.x) e[i] = __ldg(P.mesh.edges + i);
    for (int k = threadIdx.x; k < P.nkeys; k += blockDim.x) cnt[k] = 0u;
    __syncthreads();
    const size_t sec = blockIdx.y;
    const long long first = P.n * blockIdx.x / P.nblk, last = P.n * (blockIdx.x + 1) / P.nblk;
    for (long long r = first + threadIdx.x; r < last; r += blockDim.x) {
        const uint32_t key = ray_key(P, e, r);
        P.keys[sec * P.n + r] = key;
        atomicAdd(cnt + key, 1u);
    }
    __syncthreads();
    uint32_t *out = P.blk_hist + (sec * P.nblk + blockIdx.x) * (size_t)P.nkeys;
    for (int k = threadIdx.x; k < P.nkeys; k += blockDim.x) out[k] = cnt[k];
}

// per (section, key): total over the CTAs -> hist (scanned next by scan_kernel)
__global__ void __launch_bounds__(256) key_totals_kernel(const SortParams P)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= P.nkeys) return;
    const size_t sec = blockIdx.y;
    const uint32_t *in = P.blk_hist + sec * P.nblk * (size_t)P.nkeys + k;
    uint32_t t = 0;
    for (int b = 0; b < P.nblk; ++b) t += in[(size_t)b * P.nkeys];
    P.hist[sec * (P.nkeys + 1) + k] = t;
}

// per (section, key): first output position of every CTA = the key's offset + the counts of the CTAs before it
__global__ void __launch_bounds__(256) block_offsets_kernel(const SortParams P)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= P.nkeys) return;
    const size_t sec = blockIdx.y;
    uint32_t *io = P.blk_hist + sec * P.nblk * (size_t)P.nkeys + k;
    uint32_t run = P.hist[sec * (P.nkeys + 1) + k];
    for (int b0 = 0; b0 < P.nblk; b0 += 16) {          // 16 independent loads in flight, then the running sum
        uint32_t t[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) t[j] = (b0 + j < P.nblk) ? io[(size_t)(b0 + j) * P.nkeys] : 0u;
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            if (b0 + j < P.nblk) io[(size_t)(b0 + j) * P.nkeys] = run;
            run += t[j];
        }
    }
}

// dynamic shared memory: [cursors: nkeys u32]
__global__ void __launch_bounds__(1024) place_kernel(const SortParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t *cur = reinterpret_cast<uint32_t *>(smem_raw);
    const size_t sec = blockIdx.y;
    const uint32_t *in = P.blk_hist + (sec * P.nblk + blockIdx.x) * (size_t)P.nkeys;
    for (int k = threadIdx.x; k < P.nkeys; k += blockDim.x) cur[k] = in[k];
    __syncthreads();
    const long long first = P.n * blockIdx.x / P.nblk, last = P.n * (blockIdx.x + 1) / P.nblk;
    for (long long r = first + threadIdx.x; r < last; r += blockDim.x) {
        const uint32_t pos = atomicAdd(cur + P.keys[sec * P.n + r], 1u);
        P.perm[sec * P.n + pos] = (uint32_t)r;
    }
}

// one CTA per histogram (blockIdx.x = section, nkeys + 1 entries apart): exclusive prefix sum of hist[0..nkeys) in place
__global__ void __launch_bounds__(1024) scan_kernel(uint32_t *hist, int nkeys)
{
    hist += (size_t)blockIdx.x * (nkeys + 1);
    __shared__ uint32_t warp_tot[32];
    __shared__ uint32_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int first = 0; first < nkeys; first += 1024) {
        const int i = first + threadIdx.x;
        const uint32_t v = i < nkeys ? hist[i] : 0u;
        uint32_t s = v;
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += u;
        }
        if (lane == 31) warp_tot[wid] = s;
        __syncthreads();
        if (wid == 0) {
            uint32_t w = warp_tot[lane];
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, w, o);
                if (lane >= o) w += u;
            }
            warp_tot[lane] = w;
        }
        __syncthreads();
        const uint32_t before = carry + (wid ? warp_tot[wid - 1] : 0u) + (s - v);
        if (i < nkeys) hist[i] = before;
        __syncthreads();
        if (threadIdx.x == 1023) carry = before + v;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(256) scatter_kernel(const SortParams P)
{
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= P.n) return;
    const size_t sec = P.det ? blockIdx.y : 0;
    const uint32_t key = P.keys[sec * P.n + r];
    const unsigned act = __activemask();
    const unsigned peers = __match_any_sync(act, key);
    const int lane = threadIdx.x & 31, leader = __ffs(peers) - 1;
    uint32_t base = 0;
    if (lane == leader) base = atomicAdd(P.hist + sec * (P.nkeys + 1) + key, (unsigned)__popc(peers));
    base = __shfl_sync(peers, base, leader);
    const uint32_t pos = base + __popc(peers & ((1u << lane) - 1u));
    P.perm[sec * P.n + pos] = (uint32_t)r;
}

}  // namespace mr
