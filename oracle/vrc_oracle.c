/*
 * vrc_oracle.c -- CPU ORACLE for the VRC (volumetric-ray-casting) fluence estimator.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this file.
 * It shares no code, header, table or helper with the CUDA library under
 * paper_1706_07476_b200/csrc/ and neither includes the other.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md at build time of this repo):
 *   Eq. (1)  PAPER.md:23-25   F = W/S * (1 - exp(-S l))          expected path length in a cell
 *   Eq. (2)  PAPER.md:45-51   W_i = W exp(-int_0^{|r'-r|} S_t ds) attenuation to the cell entrance
 *   Eq. (3)  PAPER.md:53-56   product of the two
 *   Eq. (4)  PAPER.md:58-65   the same per ray j with weight W/N (the caller passes W/N, reading Q15)
 *   PAPER.md:85               "first calculating all cross-sections, then ray casting the particle
 *                              [through the entire geometry storing the path length travelled in each
 *                              cell], and finally calculating the VRC estimator"; cross sections are
 *                              "linearly interpolated between table values".
 * Everything is IEEE double, round-to-nearest; build with -O2 -ffp-contract=off (no FMA
 * contraction, no fast-math).  Steps O1..O6 below follow SURVEY.md §8(c) / DESIGN.md §3 in
 * that order and notation; there is no blocking, fusion or reordering.
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): numpy.interp for O2; the textbook slab
 * method for the exit parameter; brute-force sorted plane crossings for the trace; the
 * homogeneous closed form W/S(1-exp(-S L)); the collision-probability invariant; the S->0
 * track-length limit; the two-slab closed form; fine-step quadrature of the plain
 * definition; linearity, additivity and mirror symmetry; published FNV-1a test vectors.
 * The next-event function further down (vrc_next_event, steps N1..N6) is pinned in
 * tests/test_oracle_next_event_pins.py: homogeneous closed form W exp(-S R)/R^2, the void
 * inverse-square law, fine-step quadrature of Sigma_t along the line (detectors inside and outside
 * the mesh), brute-force crossing lists for the cell sequence, detectors on planes / lattice
 * points, reciprocity tau(a->b) = tau(b->a), linearity in W, every rejection rule.
 * The R-Z mesh walk (vrc_cast_rz, steps Z1..Z5) is pinned in tests/test_oracle_rz_pins.py: crossing lists from
 * numpy.roots, mid-point membership by numpy.searchsorted on (rho, z), an independent exit distance, the
 * homogeneous closed form, the collision-probability invariant, rotation invariance, quadrature.
 * Multi-nuclide materials (vrc_sigma) are pinned in tests/test_oracle_nuclide_pins.py.
 * The next-event walk on R-Z / spherical meshes (vrc_next_event_rz, steps NZ1..NZ6) is pinned in
 * tests/test_oracle_ne_rz_pins.py.  The "1/d_a not finite" branch of O1 / O4 is pinned in
 * tests/test_oracle_subnormal_pins.py.
 * Nothing in this file is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t nx, ny, nz;        /* cells per axis */
    const double *xe, *ye, *ze; /* n+1 strictly increasing plane positions per axis (cm) */
    int32_t M;                 /* materials */
    const double *density;     /* [M] g/cc */
    int32_t K;                 /* material slots per cell */
    const int32_t *cell_mat;   /* [ncell*K], -1 = empty slot; cell c = ix + nx*(iy + ny*iz) (Q17) */
    const double *cell_frac;   /* [ncell*K] volume fractions */
    const int64_t *xs_off;     /* [M+1] offsets of each material's table in xs_E / xs_sig */
    const double *xs_E;        /* energies, MeV, strictly increasing per table */
    const double *xs_sig;      /* total cross sections, cm^2/g */
    /* Multi-nuclide materials ("first calculating all cross-sections"): a
     * material m with mix_off[m+1] > mix_off[m] has no table of its own; its cross section is the weighted sum
     * of nuclide tables  sigma_m(E) = sum_j mix_w[j] * sigma_{mix_nuc[j]}(E),  j = mix_off[m] .. mix_off[m+1]-1,
     * added in that order, each nuclide table lin-lin interpolated and end-clamped like a material table.
     * N = 0 (and NULL pointers): no nuclides. */
    int32_t N;
    const int64_t *nxs_off;    /* [N+1] offsets of each nuclide's table in nxs_E / nxs_sig */
    const double *nxs_E;
    const double *nxs_sig;
    const int64_t *mix_off;    /* [M+1] */
    const int32_t *mix_nuc;    /* nuclide index per entry */
    const double *mix_w;       /* weight per entry (e.g. mass fraction: sigma stays in cm^2/g) */
} vrc_problem;

typedef struct {
    int64_t rays_accepted, rays_rejected, segments;
} vrc_counts;

/* Optional per-ray outputs (O6); any pointer may be NULL. */
typedef struct {
    uint32_t *nseg;       /* [n] segments of the ray (0 if rejected) */
    uint64_t *hash;       /* [n] FNV-1a 64 over the little-endian bytes of the uint32 cell indices, in order */
    double *sum_l;        /* [n] sum of segment lengths */
    double *t_exit;       /* [n] crossing parameter at which the ray left the mesh */
    double *tau_exit;     /* [n] optical thickness to the mesh exit */
    double *sum_score;    /* [n] sum_i score_i */
    double *sum_sig_score;/* [n] sum_i Sigma_i * score_i */
    int32_t *cells;       /* [n*cap] cell index per segment, first min(nseg,cap) filled */
    double *lens;         /* [n*cap] segment lengths */
    double *scores;       /* [n*cap] segment scores */
    int64_t cap;
} vrc_diag;

#define FNV_BASIS 0xcbf29ce484222325ULL
#define FNV_PRIME 0x100000001b3ULL

uint64_t vrc_fnv1a_cells(const uint32_t *cells, int64_t n)
{
    uint64_t h = FNV_BASIS;
    for (int64_t i = 0; i < n; ++i)
        for (int b = 0; b < 4; ++b) {
            h ^= (uint64_t)((cells[i] >> (8 * b)) & 0xffu);
            h *= FNV_PRIME;
        }
    return h;
}

/* number of elements of a[0..n) that are <= v  (std::upper_bound as an index) */
static int64_t upper_bound(const double *a, int64_t n, double v)
{
    int64_t lo = 0, hi = n;
    while (lo < hi) {
        int64_t mid = lo + (hi - lo) / 2;
        if (a[mid] <= v) lo = mid + 1; else hi = mid;
    }
    return lo;
}

/* lin-lin interpolation in one table, clamped to the end values (reading Q5) */
static double table_sigma(const double *Eg, const double *Sg, int64_t n, double E);

/* O2: sigma_m(E): the material's own table, or the weighted sum of its nuclides' tables. */
double vrc_sigma(const vrc_problem *p, int32_t m, double E)
{
    if (p->N > 0 && p->mix_off && p->mix_off[m + 1] > p->mix_off[m]) {
        double s = 0.0;
        for (int64_t j = p->mix_off[m]; j < p->mix_off[m + 1]; ++j) {
            int32_t q = p->mix_nuc[j];
            s += p->mix_w[j] * table_sigma(p->nxs_E + p->nxs_off[q], p->nxs_sig + p->nxs_off[q],
                                           p->nxs_off[q + 1] - p->nxs_off[q], E);
        }
        return s;
    }
    return table_sigma(p->xs_E + p->xs_off[m], p->xs_sig + p->xs_off[m], p->xs_off[m + 1] - p->xs_off[m], E);
}

static double table_sigma(const double *Eg, const double *Sg, int64_t n, double E)
{
    if (n == 1 || E < Eg[0]) return Sg[0];
    if (E >= Eg[n - 1]) return Sg[n - 1];
    int64_t k = upper_bound(Eg, n, E) - 1;
    if (k < 0) k = 0;
    if (k > n - 2) k = n - 2;
    double t = (E - Eg[k]) / (Eg[k + 1] - Eg[k]);
    return Sg[k] + t * (Sg[k + 1] - Sg[k]);
}

/* One ray, steps O1..O6.  Returns 1 if accepted, 0 if rejected.  tally may be NULL (trace only). */
static int cast_one(const vrc_problem *p, const double *ray, double *tally, int atomic,
                    const vrc_diag *dg, int64_t r, int64_t *segments_out)
{
    const double o[3] = {ray[0], ray[1], ray[2]};
    const double d[3] = {ray[3], ray[4], ray[5]};
    const double E = ray[6], W = ray[7];
    const int32_t n[3] = {p->nx, p->ny, p->nz};
    const double *edges[3] = {p->xe, p->ye, p->ze};

    uint32_t nseg = 0;
    uint64_t hash = FNV_BASIS;
    double sum_l = 0.0, tau = 0.0, sum_score = 0.0, sum_sig_score = 0.0, t_cur = 0.0;
    int accepted = 1;

    /* O1 validate */
    for (int f = 0; f < 8; ++f) if (!isfinite(ray[f])) accepted = 0;
    if (!(E > 0.0)) accepted = 0;
    {   /* the ray must be able to move: an axis steps only if d_a != 0 and 1/d_a is finite (Q10) */
        int movable = 0;
        for (int a = 0; a < 3; ++a) if (d[a] != 0.0 && isfinite(1.0 / d[a])) movable = 1;
        if (!movable) accepted = 0;
    }
    for (int a = 0; a < 3 && accepted; ++a)
        if (!(o[a] >= edges[a][0] && o[a] < edges[a][n[a]])) accepted = 0;

    if (accepted) {
        /* O2 cross sections of every material at the ray's energy */
        double sig[64];
        for (int32_t m = 0; m < p->M; ++m) sig[m] = vrc_sigma(p, m, E);

        /* O3 start cell: pure comparisons */
        int32_t i[3], step[3], plane[3];
        double inv[3], t[3];
        for (int a = 0; a < 3; ++a)
            i[a] = (int32_t)(upper_bound(edges[a], n[a] + 1, o[a]) - 1);

        /* O4 crossing sequences: t_a(p) = (edges_a[p] - o_a) * inv_a, one subtract then one multiply */
        for (int a = 0; a < 3; ++a) {
            inv[a] = (d[a] != 0.0) ? 1.0 / d[a] : 0.0;
            if (d[a] == 0.0 || !isfinite(inv[a])) { /* Q10: the axis never steps */
                step[a] = 0; plane[a] = 0; t[a] = INFINITY;
            } else {
                step[a] = d[a] > 0.0 ? 1 : -1;
                plane[a] = d[a] > 0.0 ? i[a] + 1 : i[a];
                t[a] = (edges[a][plane[a]] - o[a]) * inv[a];
            }
        }

        /* O5 the walk */
        for (;;) {
            int a = 0;                       /* argmin, ties x < y < z */
            if (t[1] < t[a]) a = 1;
            if (t[2] < t[a]) a = 2;
            double l = t[a] - t_cur;
            int64_t c = (int64_t)i[0] + (int64_t)n[0] * ((int64_t)i[1] + (int64_t)n[1] * (int64_t)i[2]);
            double S = 0.0;
            for (int32_t k = 0; k < p->K; ++k) {
                int32_t m = p->cell_mat[c * p->K + k];
                if (m >= 0) S += (p->cell_frac[c * p->K + k] * p->density[m]) * sig[m];
            }
            double x = S * l;
            double score = W * exp(-tau) * (x > 0.0 ? -expm1(-x) / S : l);
            if (tally) {
                if (atomic) {
#ifdef _OPENMP
#pragma omp atomic
#endif
                    tally[c] += score;
                } else
                    tally[c] += score;
            }
            if (dg && dg->cap > 0 && (int64_t)nseg < dg->cap) {
                if (dg->cells) dg->cells[r * dg->cap + nseg] = (int32_t)c;
                if (dg->lens) dg->lens[r * dg->cap + nseg] = l;
                if (dg->scores) dg->scores[r * dg->cap + nseg] = score;
            }
            for (int b = 0; b < 4; ++b) {
                hash ^= (uint64_t)(((uint32_t)c >> (8 * b)) & 0xffu);
                hash *= FNV_PRIME;
            }
            nseg += 1;
            sum_l += l;
            sum_score += score;
            sum_sig_score += S * score;
            tau += x;
            t_cur = t[a];
            i[a] += step[a];
            if (i[a] < 0 || i[a] >= n[a]) break;
            plane[a] += step[a];
            t[a] = (edges[a][plane[a]] - o[a]) * inv[a];
        }
    }

    /* O6 diagnostics */
    if (dg) {
        if (dg->nseg) dg->nseg[r] = nseg;
        if (dg->hash) dg->hash[r] = accepted ? hash : 0;
        if (dg->sum_l) dg->sum_l[r] = sum_l;
        if (dg->t_exit) dg->t_exit[r] = t_cur;
        if (dg->tau_exit) dg->tau_exit[r] = tau;
        if (dg->sum_score) dg->sum_score[r] = sum_score;
        if (dg->sum_sig_score) dg->sum_sig_score[r] = sum_sig_score;
    }
    *segments_out += nseg;
    return accepted;
}

/* Cast n rays (double AoS x,y,z,u,v,w,E,W) one after another; tally[c] += score.  Single thread. */
int vrc_cast(const vrc_problem *p, int64_t n, const double *rays, double *tally,
             const vrc_diag *dg, vrc_counts *counts)
{
    if (p->M > 64) return -1;
    vrc_counts cnt = {0, 0, 0};
    for (int64_t r = 0; r < n; ++r) {
        if (cast_one(p, rays + 8 * r, tally, 0, dg, r, &cnt.segments)) cnt.rays_accepted++;
        else cnt.rays_rejected++;
    }
    if (counts) *counts = cnt;
    return 0;
}

/* The same loop over contiguous chunks of rays on `threads` OpenMP threads.  Each thread adds into a
 * private tally when threads*ncell doubles fit in `private_bytes_max`, else all add atomically into
 * `tally`.  Private tallies are summed in thread order.  Returns the number of threads used (<0 error). */
int vrc_cast_mt(const vrc_problem *p, int64_t n, const double *rays, double *tally,
                const vrc_diag *dg, vrc_counts *counts, int threads, int64_t private_bytes_max)
{
    if (p->M > 64) return -1;
#ifndef _OPENMP
    threads = 1;
#endif
    if (threads < 1) threads = 1;
    if (threads == 1) { vrc_cast(p, n, rays, tally, dg, counts); return 1; }
    int64_t ncell = (int64_t)p->nx * p->ny * p->nz;
    int use_private = tally && (int64_t)threads * ncell * 8 <= private_bytes_max;
    double *priv = NULL;
    if (use_private) {
        priv = (double *)calloc((size_t)threads * (size_t)ncell, sizeof(double));
        if (!priv) use_private = 0;
    }
    int64_t acc = 0, rej = 0, seg = 0;
#ifdef _OPENMP
#pragma omp parallel num_threads(threads) reduction(+ : acc, rej, seg)
    {
        int tid = omp_get_thread_num();
        int nt = omp_get_num_threads();
        int64_t lo = n * tid / nt, hi = n * (tid + 1) / nt;
        double *mine = use_private ? priv + (size_t)tid * (size_t)ncell : tally;
        for (int64_t r = lo; r < hi; ++r) {
            if (cast_one(p, rays + 8 * r, mine, !use_private, dg, r, &seg)) acc++; else rej++;
        }
    }
#endif
    if (use_private) {
        for (int t = 0; t < threads; ++t)
            for (int64_t c = 0; c < ncell; ++c) tally[c] += priv[(size_t)t * (size_t)ncell + c];
        free(priv);
    }
    if (counts) { counts->rays_accepted = acc; counts->rays_rejected = rej; counts->segments = seg; }
    return threads;
}

/* ------------------------------------------------------------------------------------------------
 * Next-event (point-detector) estimator -- SURVEY.md §8(f) NEXT-3.
 *
 * "The next-event estimator (Kalos, 1963) requires a ray-cast from each source and
 * collision event to the estimator location."  The paper gives no formula; the estimator's plain
 * definition (Kalos 1963) for an event at r with weight W and a detector point r_d is
 *     score = W p(Omega_d) exp(-tau(r, r_d)) / |r_d - r|^2,   tau = int_0^R Sigma_t(r + s Omega_d, E) ds
 * with Omega_d the unit vector towards the detector and R the distance.  The caller passes the
 * weight already multiplied by the angular density p(Omega_d) (reading N-Q1, like W/N of Eq. (4)),
 * so the ray cast owes  W exp(-tau) / R^2.  Outside the mesh is void (reading N-Q2).
 *
 * Steps (all IEEE double):
 *   N1 reject (count, no contribution) an event with non-finite x,y,z,E,W, E <= 0, origin outside the
 *      half-open box, or R2 = dx*dx + dy*dy + dz*dz not finite or == 0 (d = r_d - r, one subtract per axis);
 *      the direction fields of the record are ignored
 *   N2 sigma_m(E) as O2;  N3 start cell as O3
 *   N4 crossing parameters as O4 with the UNNORMALISED direction d: t_a(p) = (edges_a[p] - o_a) * (1/d_a),
 *      so that t = 1 is the detector, exactly
 *   N5 walk as O5 (ties x<y<z); a segment whose pending crossing has t >= 1 ends AT the detector
 *      (l = 1 - t_cur) and is the last; a step that leaves the mesh is the last too.
 *      tau += Sigma_i * (l_i * R),  R = sqrt(R2)
 *   N6 score = W * exp(-tau) / R2
 * Per-event outputs: nseg, FNV-1a hash of the cell sequence, tau, score; *det_sum += score.
 * ------------------------------------------------------------------------------------------------ */
typedef struct {
    uint32_t *nseg;   /* [n] */
    uint64_t *hash;   /* [n] */
    double *tau;      /* [n] */
    double *score;    /* [n] */
} vrc_ne_diag;

static int next_event_one(const vrc_problem *p, const double *ray, const double *det, const vrc_ne_diag *dg,
                          int64_t r, double *score_out, int64_t *segments_out)
{
    const double o[3] = {ray[0], ray[1], ray[2]};
    const double E = ray[6], W = ray[7];
    const int32_t n[3] = {p->nx, p->ny, p->nz};
    const double *edges[3] = {p->xe, p->ye, p->ze};
    double d[3];
    uint32_t nseg = 0;
    uint64_t hash = FNV_BASIS;
    double tau = 0.0, score = 0.0;
    int accepted = 1;

    /* N1 */
    for (int a = 0; a < 3; ++a) if (!isfinite(o[a])) accepted = 0;
    if (!isfinite(E) || !isfinite(W) || !(E > 0.0)) accepted = 0;
    for (int a = 0; a < 3; ++a) d[a] = det[a] - o[a];
    const double R2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    if (!isfinite(R2) || !(R2 > 0.0)) accepted = 0;
    for (int a = 0; a < 3 && accepted; ++a)
        if (!(o[a] >= edges[a][0] && o[a] < edges[a][n[a]])) accepted = 0;

    if (accepted) {
        const double R = sqrt(R2);
        double sig[64];
        for (int32_t m = 0; m < p->M; ++m) sig[m] = vrc_sigma(p, m, E);        /* N2 */
        int32_t i[3], step[3], plane[3];
        double inv[3], t[3], t_cur = 0.0;
        for (int a = 0; a < 3; ++a)                                              /* N3 */
            i[a] = (int32_t)(upper_bound(edges[a], n[a] + 1, o[a]) - 1);
        for (int a = 0; a < 3; ++a) {                                            /* N4 */
            inv[a] = (d[a] != 0.0) ? 1.0 / d[a] : 0.0;
            if (d[a] == 0.0 || !isfinite(inv[a])) {
                step[a] = 0; plane[a] = 0; t[a] = INFINITY;
            } else {
                step[a] = d[a] > 0.0 ? 1 : -1;
                plane[a] = d[a] > 0.0 ? i[a] + 1 : i[a];
                t[a] = (edges[a][plane[a]] - o[a]) * inv[a];
            }
        }
        for (;;) {                                                               /* N5 */
            int a = 0;
            if (t[1] < t[a]) a = 1;
            if (t[2] < t[a]) a = 2;
            const int last = t[a] >= 1.0;
            const double l = (last ? 1.0 : t[a]) - t_cur;
            int64_t c = (int64_t)i[0] + (int64_t)n[0] * ((int64_t)i[1] + (int64_t)n[1] * (int64_t)i[2]);
            double S = 0.0;
            for (int32_t k = 0; k < p->K; ++k) {
                int32_t m = p->cell_mat[c * p->K + k];
                if (m >= 0) S += (p->cell_frac[c * p->K + k] * p->density[m]) * sig[m];
            }
            tau += S * (l * R);
            for (int b = 0; b < 4; ++b) {
                hash ^= (uint64_t)(((uint32_t)c >> (8 * b)) & 0xffu);
                hash *= FNV_PRIME;
            }
            nseg += 1;
            if (last) break;
            t_cur = t[a];
            i[a] += step[a];
            if (i[a] < 0 || i[a] >= n[a]) break;     /* the rest of the way is void (N-Q2) */
            plane[a] += step[a];
            t[a] = (edges[a][plane[a]] - o[a]) * inv[a];
        }
        score = W * exp(-tau) / R2;                                              /* N6 */
    }
    if (dg) {
        if (dg->nseg) dg->nseg[r] = nseg;
        if (dg->hash) dg->hash[r] = accepted ? hash : 0;
        if (dg->tau) dg->tau[r] = tau;
        if (dg->score) dg->score[r] = score;
    }
    *score_out = score;
    *segments_out += nseg;
    return accepted;
}

/* n events against ONE detector point det[3]; *det_sum += sum of scores (event order). */
int vrc_next_event(const vrc_problem *p, int64_t n, const double *rays, const double *det, double *det_sum,
                   const vrc_ne_diag *dg, vrc_counts *counts)
{
    if (p->M > 64) return -1;
    vrc_counts cnt = {0, 0, 0};
    double total = 0.0;
    for (int64_t r = 0; r < n; ++r) {
        double s;
        if (next_event_one(p, rays + 8 * r, det, dg, r, &s, &cnt.segments)) cnt.rays_accepted++;
        else cnt.rays_rejected++;
        total += s;
    }
    if (det_sum) *det_sum += total;
    if (counts) *counts = cnt;
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * R-Z (2-D cylindrical) tally mesh -- SURVEY.md §8(f) NEXT-4; "It must support ... 2-D
 * cylindrical (R-Z) meshes".  The paper gives no algorithm; the estimator is unchanged (Eqs. 1-4), only the
 * cells differ: cell (ir, iz) = { r_ir <= rho < r_{ir+1},  z_iz <= z < z_{iz+1} },  rho = sqrt(x^2 + y^2),
 * r_0 = 0, linear index c = ir + nr*iz.  Rays stay 3-D.
 *
 * Steps (all IEEE double, one rounding per written operation, no contraction):
 *   Z1 reject: non-finite field, E <= 0, no axis can move, rho0^2 = ox*ox + oy*oy >= r_nr*r_nr, z outside [z_0, z_nz)
 *   Z2 sigma_m(E) as O2
 *   Z3 start cell: ir = #{p in 0..nr : r_p*r_p <= rho0^2} - 1;  iz = upper_bound(z, oz) - 1
 *   Z4 radial crossings.  a = dx*dx + dy*dy, b = ox*dx + oy*dy, inv_a = 1/a; if a == 0 or inv_a is not finite
 *      the ray never crosses a cylinder.  For cylinder p:  cc_p = rho0^2 - r_p*r_p,  D_p = b*b - a*cc_p,
 *        t_in(p)  = max(0, (-b - sqrt(D_p)) * inv_a)     entering cylinder p  (shell p -> shell p-1; needs b < 0, D_p > 0)
 *        t_out(p) = max(0, (-b + sqrt(D_p)) * inv_a)     leaving cylinder p   (shell p-1 -> shell p)
 *      In shell ir the pending radial crossing is t_in(ir) while the ray still moves inward (b < 0, ir >= 1,
 *      D_ir > 0, and it has not yet turned outward), else t_out(ir+1); once outward, always outward.
 *      Axial crossings as O4:  t_z(p) = (z_p - oz) * (1/dz).
 *   Z5 walk: the pending crossing with the smaller parameter, ties radial before axial; l = t - t_cur; score as O5;
 *      an outward step from shell nr-1 or an axial step out of [0, nz) ends the ray.
 * Pins: tests/test_oracle_rz_pins.py.
 * ------------------------------------------------------------------------------------------------ */
typedef struct {
    int32_t nr, nz;
    const double *re, *ze;      /* nr+1 radii (re[0] == 0, strictly increasing), nz+1 planes */
    int32_t spherical;          /* 1: 1-D spherical shells about the origin ("1-D spherical meshes"):
                                 *    rho0^2 = ox*ox + oy*oy + oz*oz, a = dx*dx + dy*dy + dz*dz, b = ox*dx + oy*dy + oz*dz,
                                 *    no axial crossings, nz = 1 and ze is not read; everything else as Z1-Z5 */
} vrc_rz_mesh;

static int cast_one_rz(const vrc_problem *p, const vrc_rz_mesh *g, const double *ray, double *tally,
                       const vrc_diag *dg, int64_t r, int64_t *segments_out)
{
    const double ox = ray[0], oy = ray[1], oz = ray[2], dx = ray[3], dy = ray[4], dz = ray[5];
    const double E = ray[6], W = ray[7];
    const int32_t nr = g->nr, nz = g->nz;
    uint32_t nseg = 0;
    uint64_t hash = FNV_BASIS;
    double sum_l = 0.0, tau = 0.0, sum_score = 0.0, sum_sig_score = 0.0, t_cur = 0.0;
    int accepted = 1;

    /* Z1 */
    for (int f = 0; f < 8; ++f) if (!isfinite(ray[f])) accepted = 0;
    if (!(E > 0.0)) accepted = 0;
    const int sph = g->spherical != 0;
    const double rho2 = sph ? ox * ox + oy * oy + oz * oz : ox * ox + oy * oy;
    const double a = sph ? dx * dx + dy * dy + dz * dz : dx * dx + dy * dy;
    const double inv_a = (a != 0.0) ? 1.0 / a : 0.0;
    const int radial = (a != 0.0) && isfinite(inv_a) && isfinite(a);
    const double inv_z = (dz != 0.0) ? 1.0 / dz : 0.0;
    const int axial = !sph && (dz != 0.0) && isfinite(inv_z);
    if (!radial && !axial) accepted = 0;
    if (accepted && !(rho2 < g->re[nr] * g->re[nr])) accepted = 0;
    if (accepted && !sph && !(oz >= g->ze[0] && oz < g->ze[nz])) accepted = 0;

    if (accepted) {
        double sig[64];
        for (int32_t m = 0; m < p->M; ++m) sig[m] = vrc_sigma(p, m, E);         /* Z2 */
        /* Z3 */
        int32_t ir = -1;
        for (int32_t q = 0; q <= nr; ++q) if (g->re[q] * g->re[q] <= rho2) ir = q;
        int32_t iz = sph ? 0 : (int32_t)(upper_bound(g->ze, nz + 1, oz) - 1);
        /* Z4 */
        const double b = sph ? ox * dx + oy * dy + oz * dz : ox * dx + oy * dy;
        int inward = 0;
        double t_r = INFINITY, t_z = INFINITY;
        int32_t pz = 0, stepz = 0;
        if (radial) {
            if (b < 0.0 && ir >= 1) {
                double cc = rho2 - g->re[ir] * g->re[ir];
                double D = b * b - a * cc;
                if (D > 0.0) { inward = 1; t_r = fmax(0.0, (-b - sqrt(D)) * inv_a); }
            }
            if (!inward) {
                double cc = rho2 - g->re[ir + 1] * g->re[ir + 1];
                double D = b * b - a * cc;
                t_r = fmax(0.0, (-b + sqrt(D)) * inv_a);
            }
        }
        if (axial) {
            stepz = dz > 0.0 ? 1 : -1;
            pz = dz > 0.0 ? iz + 1 : iz;
            t_z = (g->ze[pz] - oz) * inv_z;
        }
        /* Z5 */
        for (;;) {
            const int ax = (t_z < t_r) ? 1 : 0;            /* ties: radial first */
            const double tn = ax ? t_z : t_r;
            double l = tn - t_cur;
            int64_t c = (int64_t)ir + (int64_t)nr * (int64_t)iz;
            double S = 0.0;
            for (int32_t k = 0; k < p->K; ++k) {
                int32_t m = p->cell_mat[c * p->K + k];
                if (m >= 0) S += (p->cell_frac[c * p->K + k] * p->density[m]) * sig[m];
            }
            double x = S * l;
            double score = W * exp(-tau) * (x > 0.0 ? -expm1(-x) / S : l);
            if (tally) tally[c] += score;
            if (dg && dg->cap > 0 && (int64_t)nseg < dg->cap) {
                if (dg->cells) dg->cells[r * dg->cap + nseg] = (int32_t)c;
                if (dg->lens) dg->lens[r * dg->cap + nseg] = l;
                if (dg->scores) dg->scores[r * dg->cap + nseg] = score;
            }
            for (int q = 0; q < 4; ++q) {
                hash ^= (uint64_t)(((uint32_t)c >> (8 * q)) & 0xffu);
                hash *= FNV_PRIME;
            }
            nseg += 1;
            sum_l += l;
            sum_score += score;
            sum_sig_score += S * score;
            tau += x;
            t_cur = tn;
            if (ax) {
                iz += stepz;
                if (iz < 0 || iz >= nz) break;
                pz += stepz;
                t_z = (g->ze[pz] - oz) * inv_z;
            } else if (inward) {
                ir -= 1;
                inward = 0;
                if (ir >= 1) {
                    double cc = rho2 - g->re[ir] * g->re[ir];
                    double D = b * b - a * cc;
                    if (D > 0.0) { inward = 1; t_r = fmax(0.0, (-b - sqrt(D)) * inv_a); }
                }
                if (!inward) {
                    double cc = rho2 - g->re[ir + 1] * g->re[ir + 1];
                    double D = b * b - a * cc;
                    t_r = fmax(0.0, (-b + sqrt(D)) * inv_a);
                }
            } else {
                ir += 1;
                if (ir >= nr) break;
                double cc = rho2 - g->re[ir + 1] * g->re[ir + 1];
                double D = b * b - a * cc;
                t_r = fmax(0.0, (-b + sqrt(D)) * inv_a);
            }
        }
    }
    if (dg) {
        if (dg->nseg) dg->nseg[r] = nseg;
        if (dg->hash) dg->hash[r] = accepted ? hash : 0;
        if (dg->sum_l) dg->sum_l[r] = sum_l;
        if (dg->t_exit) dg->t_exit[r] = t_cur;
        if (dg->tau_exit) dg->tau_exit[r] = tau;
        if (dg->sum_score) dg->sum_score[r] = sum_score;
        if (dg->sum_sig_score) dg->sum_sig_score[r] = sum_sig_score;
    }
    *segments_out += nseg;
    return accepted;
}

/* n rays on the R-Z mesh g; p supplies materials and tables (p->nx, ny, nz, xe, ye, ze are ignored; cell_mat and
 * cell_frac hold nr*nz cells).  Single thread, ray order. */
int vrc_cast_rz(const vrc_problem *p, const vrc_rz_mesh *g, int64_t n, const double *rays, double *tally,
                const vrc_diag *dg, vrc_counts *counts)
{
    if (p->M > 64 || g->nr < 1 || g->nz < 1 || g->re[0] != 0.0 || (g->spherical && g->nz != 1)) return -1;
    vrc_counts cnt = {0, 0, 0};
    for (int64_t r = 0; r < n; ++r) {
        if (cast_one_rz(p, g, rays + 8 * r, tally, dg, r, &cnt.segments)) cnt.rays_accepted++;
        else cnt.rays_rejected++;
    }
    if (counts) *counts = cnt;
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Next-event (point-detector) estimator on R-Z and spherical meshes -- the NEXT-3 x NEXT-4 cell of SURVEY.md §8(f)
 * ("requires a ray-cast from each source and collision event to the estimator location"; PAPER.md:358
 * "1-D spherical ... 2-D cylindrical (R-Z) meshes").  The estimator is that of vrc_next_event, the cells those of
 * vrc_cast_rz; nothing new is read into the paper (readings N-Q1..N-Q6 and Z-Q1..Z-Q5 of DESIGN.md §10 apply).
 *
 * Steps (all IEEE double, one rounding per written operation):
 *   NZ1 reject (count, no contribution) an event with non-finite x, y, z, E or W, E <= 0, rho0^2 >= r_nr^2, z outside
 *       [z_0, z_nz) (R-Z only), or, with d = det - o (one subtract per axis), R2 = dx*dx + dy*dy + dz*dz not finite or
 *       == 0, or no crossing family that can move (Z1: a == 0 or 1/a not finite, and dz == 0 or 1/dz not finite);
 *       the direction fields of the record are ignored
 *   NZ2 sigma_m(E) as O2;   NZ3 start cell as Z3
 *   NZ4 crossing parameters as Z4 with the UNNORMALISED direction d, so that t = 1 is the detector, exactly
 *   NZ5 walk as Z5 (ties radial before axial); a segment whose pending crossing has t >= 1 ends AT the detector
 *       (l = 1 - t_cur) and is the last; a step that leaves the mesh is the last too (outside is void, N-Q2).
 *       tau += Sigma_i * (l_i * R),  R = sqrt(R2)
 *   NZ6 score = W * exp(-tau) / R2
 * Pins: tests/test_oracle_ne_rz_pins.py (homogeneous closed form, void inverse-square law, numpy.roots crossing lists
 * cut at t = 1, quadrature of Sigma_t along the line, detectors on cylinders / planes / the axis, reciprocity,
 * rotation invariance, every rejection rule).
 * ------------------------------------------------------------------------------------------------ */
static int next_event_rz_one(const vrc_problem *p, const vrc_rz_mesh *g, const double *ray, const double *det,
                             const vrc_ne_diag *dg, int64_t r, double *score_out, int64_t *segments_out)
{
    const double ox = ray[0], oy = ray[1], oz = ray[2];
    const double E = ray[6], W = ray[7];
    const int32_t nr = g->nr, nz = g->nz;
    const int sph = g->spherical != 0;
    uint32_t nseg = 0;
    uint64_t hash = FNV_BASIS;
    double tau = 0.0, score = 0.0;
    int accepted = 1;

    /* NZ1 */
    if (!isfinite(ox) || !isfinite(oy) || !isfinite(oz) || !isfinite(E) || !isfinite(W) || !(E > 0.0)) accepted = 0;
    const double dx = det[0] - ox, dy = det[1] - oy, dz = det[2] - oz;
    const double R2 = dx * dx + dy * dy + dz * dz;
    if (!isfinite(R2) || !(R2 > 0.0)) accepted = 0;
    const double rho2 = sph ? ox * ox + oy * oy + oz * oz : ox * ox + oy * oy;
    const double a = sph ? dx * dx + dy * dy + dz * dz : dx * dx + dy * dy;
    const double inv_a = (a != 0.0) ? 1.0 / a : 0.0;
    const int radial = (a != 0.0) && isfinite(inv_a) && isfinite(a);
    const double inv_z = (dz != 0.0) ? 1.0 / dz : 0.0;
    const int axial = !sph && (dz != 0.0) && isfinite(inv_z);
    if (!radial && !axial) accepted = 0;
    if (accepted && !(rho2 < g->re[nr] * g->re[nr])) accepted = 0;
    if (accepted && !sph && !(oz >= g->ze[0] && oz < g->ze[nz])) accepted = 0;

    if (accepted) {
        const double R = sqrt(R2);
        double sig[64];
        for (int32_t m = 0; m < p->M; ++m) sig[m] = vrc_sigma(p, m, E);         /* NZ2 */
        /* NZ3 */
        int32_t ir = -1;
        for (int32_t q = 0; q <= nr; ++q) if (g->re[q] * g->re[q] <= rho2) ir = q;
        int32_t iz = sph ? 0 : (int32_t)(upper_bound(g->ze, nz + 1, oz) - 1);
        /* NZ4 */
        const double b = sph ? ox * dx + oy * dy + oz * dz : ox * dx + oy * dy;
        int inward = 0;
        double t_r = INFINITY, t_z = INFINITY, t_cur = 0.0;
        int32_t pz = 0, stepz = 0;
        if (radial) {
            if (b < 0.0 && ir >= 1) {
                double cc = rho2 - g->re[ir] * g->re[ir];
                double D = b * b - a * cc;
                if (D > 0.0) { inward = 1; t_r = fmax(0.0, (-b - sqrt(D)) * inv_a); }
            }
            if (!inward) {
                double cc = rho2 - g->re[ir + 1] * g->re[ir + 1];
                double D = b * b - a * cc;
                t_r = fmax(0.0, (-b + sqrt(D)) * inv_a);
            }
        }
        if (axial) {
            stepz = dz > 0.0 ? 1 : -1;
            pz = dz > 0.0 ? iz + 1 : iz;
            t_z = (g->ze[pz] - oz) * inv_z;
        }
        /* NZ5 */
        for (;;) {
            const int ax = (t_z < t_r) ? 1 : 0;            /* ties: radial first */
            const double tn = ax ? t_z : t_r;
            const int last = tn >= 1.0;
            const double l = (last ? 1.0 : tn) - t_cur;
            int64_t c = (int64_t)ir + (int64_t)nr * (int64_t)iz;
            double S = 0.0;
            for (int32_t k = 0; k < p->K; ++k) {
                int32_t m = p->cell_mat[c * p->K + k];
                if (m >= 0) S += (p->cell_frac[c * p->K + k] * p->density[m]) * sig[m];
            }
            tau += S * (l * R);
            for (int q = 0; q < 4; ++q) {
                hash ^= (uint64_t)(((uint32_t)c >> (8 * q)) & 0xffu);
                hash *= FNV_PRIME;
            }
            nseg += 1;
            if (last) break;
            t_cur = tn;
            if (ax) {
                iz += stepz;
                if (iz < 0 || iz >= nz) break;
                pz += stepz;
                t_z = (g->ze[pz] - oz) * inv_z;
            } else if (inward) {
                ir -= 1;
                inward = 0;
                if (ir >= 1) {
                    double cc = rho2 - g->re[ir] * g->re[ir];
                    double D = b * b - a * cc;
                    if (D > 0.0) { inward = 1; t_r = fmax(0.0, (-b - sqrt(D)) * inv_a); }
                }
                if (!inward) {
                    double cc = rho2 - g->re[ir + 1] * g->re[ir + 1];
                    double D = b * b - a * cc;
                    t_r = fmax(0.0, (-b + sqrt(D)) * inv_a);
                }
            } else {
                ir += 1;
                if (ir >= nr) break;
                double cc = rho2 - g->re[ir + 1] * g->re[ir + 1];
                double D = b * b - a * cc;
                t_r = fmax(0.0, (-b + sqrt(D)) * inv_a);
            }
        }
        score = W * exp(-tau) / R2;                                              /* NZ6 */
    }
    if (dg) {
        if (dg->nseg) dg->nseg[r] = nseg;
        if (dg->hash) dg->hash[r] = accepted ? hash : 0;
        if (dg->tau) dg->tau[r] = tau;
        if (dg->score) dg->score[r] = score;
    }
    *score_out = score;
    *segments_out += nseg;
    return accepted;
}

/* n events against ONE detector point det[3] on the R-Z / spherical mesh g; *det_sum += sum of scores (event order). */
int vrc_next_event_rz(const vrc_problem *p, const vrc_rz_mesh *g, int64_t n, const double *rays, const double *det,
                      double *det_sum, const vrc_ne_diag *dg, vrc_counts *counts)
{
    if (p->M > 64 || g->nr < 1 || g->nz < 1 || g->re[0] != 0.0 || (g->spherical && g->nz != 1)) return -1;
    vrc_counts cnt = {0, 0, 0};
    double total = 0.0;
    for (int64_t r = 0; r < n; ++r) {
        double s;
        if (next_event_rz_one(p, g, rays + 8 * r, det, dg, r, &s, &cnt.segments)) cnt.rays_accepted++;
        else cnt.rays_rejected++;
        total += s;
    }
    if (det_sum) *det_sum += total;
    if (counts) *counts = cnt;
    return 0;
}

int vrc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
