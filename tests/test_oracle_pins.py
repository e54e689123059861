"""Pins for the CPU oracle (oracle/vrc_oracle.c) against things OTHER than itself.

Each test names what fixes the expected value: a library routine, a textbook method, a closed
form, an invariant, brute force, or quadrature of the plain definition
    score_i = W * int_{s in cell i} exp(-tau(s)) ds,  tau(s) = int_0^s Sigma_t ds'
(PAPER.md:23-25 Eq. 1, :45-56 Eqs. 2-3, :58-65 Eq. 4).  The paper prints no worked numerical
example, so there is no paper-value fixture.
"""
import numpy as np
import pytest

from oracle.vrc_oracle import Oracle, fnv1a_cells
from tests.tiny import tiny_problem, tiny_rays
from workloads import make_problem, make_rays


# ----------------------------------------------------------------------------- independent helpers
def np_sigma_cell(prob, E):
    """Sigma_t of every cell at energy E from numpy.interp (library lin-lin interpolation with end clamping)."""
    sig = np.array([np.interp(E, e, s) for e, s in prob.xs])
    S = np.zeros(prob.ncell)
    for k in range(prob.K):
        m = prob.cell_mat[:, k]
        S += np.where(m >= 0, prob.cell_frac[:, k] * prob.density[np.maximum(m, 0)] * sig[np.maximum(m, 0)], 0.0)
    return S


def slab_exit(prob, o, d):
    """Textbook slab-method exit parameter of a ray that starts inside an axis-aligned box."""
    t = np.inf
    for a, e in enumerate((prob.xe, prob.ye, prob.ze)):
        if d[a] > 0:
            t = min(t, (e[-1] - o[a]) * (1.0 / d[a]))
        elif d[a] < 0:
            t = min(t, (e[0] - o[a]) * (1.0 / d[a]))
    return t


def brute_trace(prob, o, d):
    """All plane crossings of the ray, stable-sorted by (t, axis); cells visited until the mesh is left."""
    edges = (prob.xe, prob.ye, prob.ze)
    n = (prob.nx, prob.ny, prob.nz)
    idx = [int(np.searchsorted(edges[a], o[a], side="right")) - 1 for a in range(3)]
    ev = []
    for a in range(3):
        if d[a] == 0:
            continue
        inv = 1.0 / d[a]
        planes = range(idx[a] + 1, n[a] + 1) if d[a] > 0 else range(idx[a], -1, -1)
        for seq, p in enumerate(planes):
            ev.append(((edges[a][p] - o[a]) * inv, a, seq))
    ev.sort()
    cells, lens, t_cur = [], [], 0.0
    for t, a, _ in ev:
        cells.append(idx[0] + n[0] * (idx[1] + n[1] * idx[2]))
        lens.append(t - t_cur)
        t_cur = t
        idx[a] += 1 if d[a] > 0 else -1
        if idx[a] < 0 or idx[a] >= n[a]:
            break
    return np.array(cells), np.array(lens), t_cur


def py_fnv1a(data: bytes) -> int:
    h = 0xCBF29CE484222325
    for b in data:
        h = ((h ^ b) * 0x100000001B3) & 0xFFFFFFFFFFFFFFFF
    return h


# ----------------------------------------------------------------------------- O2 cross sections
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_sigma_equals_numpy_interp(seed):
    """PAPER.md:85 'linearly interpolated between table values' == numpy.interp (clamps at both ends)."""
    prob = tiny_problem(seed, n_e=40)
    orc = Oracle(prob)
    g = np.random.default_rng(seed)
    for m, (e, s) in enumerate(prob.xs):
        probe = np.concatenate([e, 0.5 * (e[1:] + e[:-1]), [e[0] * 0.5, e[-1] * 2.0, e[0], e[-1]],
                                e[0] * (e[-1] / e[0]) ** g.random(200)])
        got = np.array([orc.sigma(m, x) for x in probe])
        want = np.interp(probe, e, s)
        np.testing.assert_allclose(got, want, rtol=1e-13, atol=0)  # numpy rounds slope*(x-x0): a few ulp
        # exact table values at grid points; exact mid-point average (both sums are exact in double for fp32 data)
        assert np.array_equal(got[: len(e)], s)


def test_sigma_on_config_tables():
    prob = make_problem(1)
    orc = Oracle(prob)
    g = np.random.default_rng(0)
    for m, (e, s) in enumerate(prob.xs):
        probe = 1e-12 * (1e14) ** g.random(500)
        got = np.array([orc.sigma(m, x) for x in probe])
        np.testing.assert_allclose(got, np.interp(probe, e, s), rtol=1e-13)


# ----------------------------------------------------------------------------- trace
@pytest.mark.parametrize("seed,uniform", [(11, False), (12, True), (13, False)])
def test_trace_equals_brute_force(seed, uniform):
    """The 3-way merge equals a stable sort of every plane crossing by (t, axis) -- SURVEY.md §8(c) O4."""
    prob = tiny_problem(seed, nx=5, ny=4, nz=6, uniform=uniform)
    orc = Oracle(prob)
    rays = tiny_rays(prob, seed, 300, axis_aligned_share=0.2)
    cap = prob.nx + prob.ny + prob.nz + 3
    res = orc.cast(rays, cap=cap)
    assert res.rays_rejected == 0
    for r in range(len(rays)):
        o, d = rays[r, :3].astype(np.float64), rays[r, 3:6].astype(np.float64)
        cells, lens, t_exit = brute_trace(prob, o, d)
        assert res.nseg[r] == len(cells)
        assert np.array_equal(res.cells[r, : len(cells)], cells)
        assert np.array_equal(res.lens[r, : len(cells)], lens)  # same double expressions -> bitwise
        assert res.t_exit[r] == t_exit
        assert res.hash[r] == py_fnv1a(cells.astype("<u4").tobytes())


def test_trace_on_lattice_points_and_corners():
    """Edge and corner hits: ties resolve x<y<z, one axis per step, zero-length segments kept (Q9)."""
    prob = tiny_problem(21, nx=4, ny=4, nz=4, uniform=True)
    orc = Oracle(prob)
    # origins on lattice planes / cell corners, directions along diagonals: exact ties in t
    rays = []
    for o in ([-1.0, -1.0, -1.0], [-0.25, -0.25, 0.5], [0.5, -0.25, -0.25], [-1.0, 0.5, 1.25]):
        for d in ([1, 1, 1], [1, 1, 0], [-1, 1, 1], [1, -1, -1], [0, 0, 1], [-1, -1, -1], [2, 1, 1]):
            rays.append(o + d + [1.0, 1.0])
    rays = np.array(rays, dtype=np.float64)
    res = orc.cast(rays, cap=16)
    assert res.rays_rejected == 0
    for r in range(len(rays)):
        cells, lens, t_exit = brute_trace(prob, rays[r, :3], rays[r, 3:6])
        assert res.nseg[r] == len(cells)
        assert np.array_equal(res.cells[r, : len(cells)], cells)
        assert np.array_equal(res.lens[r, : len(cells)], lens)
    # the all-ones diagonal from the low corner: x, y, z cross together -> two zero-length segments per lattice point
    cells, lens, _ = brute_trace(prob, rays[0, :3], rays[0, 3:6])
    assert (lens == 0).sum() == 2 * 3 and len(cells) == 3 * 4 - 2  # leaves on the 4th x crossing, before its y and z ties


def test_axis_aligned_segment_count_and_length():
    """An axis-aligned ray crosses n - i0 cells of length h (SURVEY.md §8(c) pins)."""
    prob = tiny_problem(5, nx=7, ny=3, nz=2, uniform=True)
    orc = Oracle(prob)
    h = 0.75
    o = [-1.0 + 2.3 * h, -1.0 + 1.5 * h, -1.0 + 0.5 * h]
    res = orc.cast(np.array([o + [1, 0, 0, 1.0, 1.0], o + [-1, 0, 0, 1.0, 1.0], o + [0.0, -0.0, 1, 1.0, 1.0]]), cap=8)
    assert list(res.nseg) == [7 - 2, 3, 2]
    np.testing.assert_allclose(res.lens[0, 1:5], h, rtol=1e-15)
    np.testing.assert_allclose(res.lens[0, 0], 0.7 * h, rtol=1e-14)
    assert list(res.cells[1, :3]) == [2 + 7 * 1, 1 + 7 * 1, 0 + 7 * 1]


@pytest.mark.parametrize("cfg", [1, 3])
def test_exit_parameter_is_the_slab_method_bitwise(cfg):
    """Last crossing parameter == slab-method box exit written with (edge - o) * inv; sum l == t_exit."""
    prob = make_problem(cfg) if cfg == 1 else make_problem(3, nx=34, ny=34, nz=20, n_e=500)
    orc = Oracle(prob)
    rays = make_rays(prob, 2000)
    res = orc.cast(rays, per_ray=True)
    for r in range(len(rays)):
        t = slab_exit(prob, rays[r, :3].astype(np.float64), rays[r, 3:6].astype(np.float64))
        assert res.t_exit[r] == t
        assert abs(res.sum_l[r] - t) <= res.nseg[r] * 2.0**-52 * t


# ----------------------------------------------------------------------------- scores
def test_homogeneous_closed_form():
    """One material everywhere: sum_i score_i = W/S (1 - exp(-S L)) (telescoping of Eq. 3; north_star)."""
    prob = tiny_problem(31, nx=6, ny=5, nz=4, homogeneous=True)
    orc = Oracle(prob)
    rays = tiny_rays(prob, 31, 500)
    res = orc.cast(rays, per_ray=True)
    for r in range(len(rays)):
        E, W = float(rays[r, 6]), float(rays[r, 7])
        S = prob.density[0] * np.interp(E, *prob.xs[0])
        L = slab_exit(prob, rays[r, :3].astype(np.float64), rays[r, 3:6].astype(np.float64))
        want = W / S * (1.0 - np.exp(-S * L))
        assert res.sum_score[r] == pytest.approx(want, rel=1e-13)
        assert res.tau_exit[r] == pytest.approx(S * L, rel=1e-13)
    assert res.tally.sum() == pytest.approx(res.sum_score.sum(), rel=1e-13)


def test_collision_probability_invariant():
    """Any medium: sum_i Sigma_i score_i = W (1 - exp(-tau_exit)), with tau_exit from numpy-side sums."""
    prob = tiny_problem(41, nx=6, ny=6, nz=6, K=3)
    orc = Oracle(prob)
    rays = tiny_rays(prob, 41, 400)
    res = orc.cast(rays, cap=32)
    for r in range(len(rays)):
        E, W = float(rays[r, 6]), float(rays[r, 7])
        S = np_sigma_cell(prob, E)
        n = res.nseg[r]
        tau = float(np.sum(S[res.cells[r, :n]] * res.lens[r, :n]))
        assert res.tau_exit[r] == pytest.approx(tau, rel=1e-13)
        assert res.sum_sig_score[r] == pytest.approx(W * (1.0 - np.exp(-tau)), rel=1e-12)
        # and score by score against the closed form with numpy's own Sigma and running optical depth
        t_in = np.concatenate([[0.0], np.cumsum(S[res.cells[r, :n]] * res.lens[r, :n])[:-1]])
        Sc = S[res.cells[r, :n]]
        with np.errstate(divide="ignore", invalid="ignore"):
            want = np.where(Sc > 0, W * (np.exp(-t_in) - np.exp(-t_in - Sc * res.lens[r, :n])) / Sc,
                                W * np.exp(-t_in) * res.lens[r, :n])
        np.testing.assert_allclose(res.scores[r, :n], want, rtol=1e-9, atol=1e-15)


def test_void_limit_is_the_track_length():
    """All densities 0 => score_i = W l_i exactly and sum tally = sum_rays W L (Eq. 1 limit, Q12)."""
    prob = tiny_problem(51, void=True)
    orc = Oracle(prob)
    rays = tiny_rays(prob, 51, 300)
    res = orc.cast(rays, cap=16)
    total = 0.0
    for r in range(len(rays)):
        n = res.nseg[r]
        assert np.array_equal(res.scores[r, :n], float(rays[r, 7]) * res.lens[r, :n])
        total += float(rays[r, 7]) * slab_exit(prob, rays[r, :3].astype(np.float64), rays[r, 3:6].astype(np.float64))
    assert res.tally.sum() == pytest.approx(total, rel=1e-13)


def test_two_slab_closed_form_config1():
    """Config 1, rays along +-z through the concrete (z<3) / air interface: antiderivative differences."""
    prob = make_problem(1)
    orc = Oracle(prob)
    E, W = 0.7, 1.25
    Sa = prob.density[0] * np.interp(E, *prob.xs[0])
    Sc = prob.density[1] * np.interp(E, *prob.xs[1])

    def tau_at(z0, z1):  # optical depth between heights z0 <= z1
        conc = max(0.0, min(z1, 3.0) - min(z0, 3.0))
        return Sc * conc + Sa * ((z1 - z0) - conc)

    for z0, sgn in ((0.5, +1), (9.25, -1), (2.999, +1), (3.0, -1)):
        ray = np.array([[4.5, 6.5, z0, 0.0, 0.0, float(sgn), E, W]])
        res = orc.cast(ray)
        col = res.tally.reshape(10, 10, 10)[:, 6, 4]
        for iz in range(10):
            a, b = (max(iz, z0), iz + 1) if sgn > 0 else (iz, min(iz + 1, z0))
            if b <= a and not (sgn < 0 and z0 == iz):
                assert col[iz] == 0.0
                continue
            S = Sc if iz < 3 else Sa
            if sgn > 0:
                want = W / S * (np.exp(-tau_at(z0, a)) - np.exp(-tau_at(z0, b)))
            else:
                want = W / S * (np.exp(-tau_at(b, z0)) - np.exp(-tau_at(a, z0)))
            assert col[iz] == pytest.approx(want, rel=1e-9, abs=1e-300)
        assert res.tally.sum() == pytest.approx(col.sum(), rel=1e-15)


@pytest.mark.parametrize("seed", [61, 62])
def test_quadrature_of_the_plain_definition(seed):
    """Mid-point quadrature of W int exp(-tau(s)) ds along each ray, cells located by searchsorted."""
    prob = tiny_problem(seed, nx=4, ny=3, nz=5, K=2)
    orc = Oracle(prob)
    rays = tiny_rays(prob, seed, 12).astype(np.float64)
    N = 400_000
    for r in range(len(rays)):
        o, d, E, W = rays[r, :3], rays[r, 3:6], rays[r, 6], rays[r, 7]
        L = slab_exit(prob, o, d)
        ds = L / N
        s = (np.arange(N) + 0.5) * ds
        pos = o[None, :] + s[:, None] * d[None, :]
        ix = np.clip(np.searchsorted(prob.xe, pos[:, 0], side="right") - 1, 0, prob.nx - 1)
        iy = np.clip(np.searchsorted(prob.ye, pos[:, 1], side="right") - 1, 0, prob.ny - 1)
        iz = np.clip(np.searchsorted(prob.ze, pos[:, 2], side="right") - 1, 0, prob.nz - 1)
        c = ix + prob.nx * (iy + prob.ny * iz)
        S = np_sigma_cell(prob, E)[c]
        tau_mid = np.cumsum(S * ds) - 0.5 * S * ds
        want = np.bincount(c, weights=W * np.exp(-tau_mid) * ds, minlength=prob.ncell)
        got = orc.cast(rays[r : r + 1]).tally
        assert np.abs(got - want).max() <= 2e-4 * want.max()
        assert got.sum() == pytest.approx(want.sum(), rel=1e-5)
        assert set(np.flatnonzero(got)) >= set(np.flatnonzero(want > 1e-9 * want.max()))


# ----------------------------------------------------------------------------- linearity, additivity, symmetry
def test_linearity_additivity_mirror():
    prob = tiny_problem(71, nx=5, ny=4, nz=3, K=2)
    orc = Oracle(prob)
    rays = tiny_rays(prob, 71, 200).astype(np.float64)
    base = orc.cast(rays).tally
    dbl = rays.copy()
    dbl[:, 7] *= 2.0
    assert np.array_equal(orc.cast(dbl).tally, 2.0 * base)  # doubling W doubles every score exactly
    neg = rays.copy()
    neg[:, 7] *= -1.0
    assert np.array_equal(orc.cast(neg).tally, -base)  # Q19: any finite weight
    t = orc.cast(rays[:77]).tally
    orc.cast(rays[77:], tally=t)
    np.testing.assert_allclose(t, base, rtol=1e-13, atol=0)
    # mirror x: edges -> -edges reversed, cells flipped in x, rays x -> -x, u -> -u
    from types import SimpleNamespace
    cm = prob.cell_mat.reshape(prob.nz, prob.ny, prob.nx, prob.K)[:, :, ::-1].reshape(-1, prob.K)
    cf = prob.cell_frac.reshape(prob.nz, prob.ny, prob.nx, prob.K)[:, :, ::-1].reshape(-1, prob.K)
    mp = SimpleNamespace(**{**prob.__dict__, "xe": -prob.xe[::-1], "cell_mat": cm, "cell_frac": cf})
    mr = rays.copy()
    mr[:, 0] *= -1.0
    mr[:, 3] *= -1.0
    mt = Oracle(mp).cast(mr).tally.reshape(prob.nz, prob.ny, prob.nx)[:, :, ::-1].reshape(-1)
    np.testing.assert_allclose(mt, base, rtol=1e-13, atol=0)


# ----------------------------------------------------------------------------- O1 rejection, hash
def test_rejection_rules():
    prob = tiny_problem(81, uniform=True)  # box [-1, 2] x [-1, 1.25] x [-1, 2.75]
    orc = Oracle(prob)
    ok = [0.0, 0.0, 0.0, 0.6, 0.0, 0.8, 1.0, 1.0]
    bad = []
    for f, v in ((0, np.nan), (4, np.inf), (6, 0.0), (6, -1.0), (7, np.nan), (0, 2.0), (1, -1.0000001), (2, 2.75)):
        b = list(ok)
        b[f] = v
        bad.append(b)
    bad.append([0.0, 0.0, 0.0, 0.0, -0.0, 0.0, 1.0, 1.0])  # zero direction
    lowface = [-1.0, -1.0, -1.0, 0.6, 0.0, 0.8, 1.0, 1.0]  # on the lower faces: inside (half-open box)
    res = orc.cast(np.array([ok] + bad + [lowface]), per_ray=True)
    assert res.rays_accepted == 2 and res.rays_rejected == len(bad)
    assert np.all(res.nseg[1:-1] == 0) and res.nseg[0] > 0 and res.nseg[-1] > 0
    only = orc.cast(np.array([ok, lowface]))
    assert np.array_equal(res.tally, only.tally)


def test_fnv1a_published_vectors():
    """FNV-1a 64: offset basis for the empty string and the published vectors for 'a' and 'foobar'."""
    assert py_fnv1a(b"") == 0xCBF29CE484222325
    assert py_fnv1a(b"a") == 0xAF63DC4C8601EC8C
    assert py_fnv1a(b"foobar") == 0x85944171F73967E8
    g = np.random.default_rng(3)
    cells = g.integers(0, 2**31, size=1000).astype(np.uint32)
    assert fnv1a_cells(cells) == py_fnv1a(cells.astype("<u4").tobytes())
    assert fnv1a_cells(cells[:0]) == 0xCBF29CE484222325
    # 'foob' as one little-endian word then 'ar..': prefix property on whole words
    w = np.frombuffer(b"foobarba", dtype="<u4")
    assert fnv1a_cells(w) == py_fnv1a(b"foobarba")


def test_multithreaded_equals_single():
    prob = make_problem(1)
    orc = Oracle(prob)
    rays = make_rays(prob, 5000)
    a = orc.cast(rays, per_ray=True)
    b = orc.cast(rays, per_ray=True, threads=4)
    assert np.array_equal(a.nseg, b.nseg) and np.array_equal(a.hash, b.hash) and a.segments == b.segments
    np.testing.assert_allclose(b.tally, a.tally, rtol=1e-13)
    c = orc.cast(rays, threads=4, private_bytes_max=0)  # atomic-add branch
    np.testing.assert_allclose(c.tally, a.tally, rtol=1e-13)
