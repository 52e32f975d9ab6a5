"""Pins of the oracle's droplet analysis, second stage (PAPER section 2.4 L198-200 and Eq. (25); readings
R23-R26 of DESIGN.md): digital Voronoi colouring, Delaunay links from the Voronoi vertices, droplet matching and T1
events between two frames, droplet Nusselt number.  No GPU, no CUDA path.

The expected values come from hand-made cases, from the defining property written out in numpy, from
scipy.spatial's continuum Delaunay triangulation (a library routine the digital construction must reduce to on
non-degenerate arrangements) and from closed forms."""
import itertools

import numpy as np
import pytest
from scipy.spatial import Delaunay

_CX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1], dtype=np.float64)[:, None, None]
_CY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1], dtype=np.float64)[:, None, None]
_WQ = np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)[:, None, None]


def _linear_pops(dens, ux, uy):
    return _WQ * dens * (1 + 3 * (_CX * ux + _CY * uy))


# ---------------------------------------------------------------- R23: digital Voronoi tessellation

def test_voronoi_half_planes_seam_and_ties(oracle_mod):
    """Two centres on one row: the cell boundary is the perpendicular bisector, across the periodic seam too; a
    site at equal distance from both goes to the smaller index (R23)."""
    nx, ny = 16, 6
    col = oracle_mod.voronoi(nx, ny, 0, [[2.0, 2.5], [6.0, 2.5]])
    # distances along x: site 4 is 2 from both (tie -> 0); sites 5..11 nearer to centre 1 (site 12: 6 from both
    # through the seam -> tie -> 0); sites 13..15, 0..3 nearer to centre 0
    expect = np.array([0, 0, 0, 0, 0, 1, 1, 1, 1, 1, 1, 1, 0, 0, 0, 0], dtype=np.int32)
    assert (col == expect[None, :]).all()
    # swapping the order of the centres swaps the colours except at the ties
    col2 = oracle_mod.voronoi(nx, ny, 0, [[6.0, 2.5], [2.0, 2.5]])
    expect2 = 1 - expect
    expect2[[4, 12]] = 0
    assert (col2 == expect2[None, :]).all()
    assert (oracle_mod.voronoi(nx, ny, 0, np.zeros((0, 2))) == -1).all()


def test_voronoi_rectangular_cells(oracle_mod):
    """Centres at the middles of the boxes of a regular gx x gy partition: every box is exactly one cell."""
    nx, ny, gx, gy = 40, 24, 5, 3
    bx, by = nx // gx, ny // gy
    centres = [[(i + 0.5) * bx - 0.5, (j + 0.5) * by - 0.5] for j in range(gy) for i in range(gx)]
    expect = (np.arange(ny)[:, None] // by) * gx + np.arange(nx)[None, :] // bx
    for per in (0, 1):
        assert (oracle_mod.voronoi(nx, ny, per, centres) == expect).all()


def test_voronoi_y_wraps_only_when_periodic(oracle_mod):
    nx, ny = 8, 20
    centres = [[4.0, 1.0], [4.0, 9.0]]
    walls = oracle_mod.voronoi(nx, ny, 0, centres)
    per = oracle_mod.voronoi(nx, ny, 1, centres)
    assert (walls[19] == 1).all()  # |19 - 9| = 10 < |19 - 1| = 18
    assert (per[19] == 0).all()    # through the seam: 2 < 10
    assert (walls[:5] == per[:5]).all() and (walls[:5] == 0).all()


@pytest.mark.parametrize("per", [0, 1])
def test_voronoi_defining_minimum_property(oracle_mod, per):
    """colour = the index with the smallest minimum-image distance, first index on ties -- the definition written
    out with numpy broadcasting on random centres."""
    rng = np.random.default_rng(5 + per)
    nx, ny, n = 37, 23, 17
    c = rng.random((n, 2)) * [nx, ny]
    col = oracle_mod.voronoi(nx, ny, per, c)
    X, Y = np.meshgrid(np.arange(nx, dtype=np.float64), np.arange(ny, dtype=np.float64))
    dx = X[None] - c[:, 0, None, None]
    dx = np.where(dx > nx / 2, dx - nx, np.where(dx < -nx / 2, dx + nx, dx))
    dy = Y[None] - c[:, 1, None, None]
    if per:
        dy = np.where(dy > ny / 2, dy - ny, np.where(dy < -ny / 2, dy + ny, dy))
    assert (col == np.argmin(dx * dx + dy * dy, axis=0)).all()


# ---------------------------------------------------------------- R24: Delaunay links

def _triangular_arrangement(nx, ny, cols, rows, jitter, seed, y_margin=0.0):
    """cols x rows centres on a triangular lattice filling [0, nx) x [y_margin, ny - y_margin), jittered."""
    rng = np.random.default_rng(seed)
    ax, ay = nx / cols, (ny - 2 * y_margin) / rows
    pts = []
    for j in range(rows):
        for i in range(cols):
            pts.append([(i + 0.5 * (j % 2) + 0.25) * ax, y_margin + (j + 0.5) * ay])
    pts = np.array(pts) + (rng.random((cols * rows, 2)) - 0.5) * jitter
    pts[:, 0] %= nx
    return pts


def _continuum_links(pts, nx, ny, periodic_y):
    """Links of the continuum Delaunay triangulation of the centres on the x-periodic strip: periodic images in x
    (and in y when periodic); between walls the mirror images beyond y = -1/2 and y = ny - 1/2, so that two cells
    sharing a Voronoi edge that ends on a wall stay neighbours (their link is the convex-hull edge the wall colour
    of R24 stands for).  A link counts if it joins two different real droplets through any image."""
    n = len(pts)
    allp, owner, real = [], [], []
    for sx in (-1, 0, 1):
        ys = (-1, 0, 1) if periodic_y else (0,)
        for sy in ys:
            allp.append(pts + [sx * nx, sy * ny])
            owner.append(np.arange(n))
            real.append(np.full(n, sx == 0 and sy == 0))
        if not periodic_y:
            for mirror in (-1.0 - pts[:, 1], 2.0 * ny - 1.0 - pts[:, 1]):  # reflections in the wall planes
                allp.append(np.stack([pts[:, 0] + sx * nx, mirror], 1))
                owner.append(np.full(n, -1))
                real.append(np.full(n, False))
    allp, owner, real = np.concatenate(allp), np.concatenate(owner), np.concatenate(real)
    tri = Delaunay(allp)
    out = set()
    for s in tri.simplices:
        for a, b in itertools.combinations(s, 2):
            if (real[a] or real[b]) and owner[a] >= 0 and owner[b] >= 0 and owner[a] != owner[b]:
                out.add((min(owner[a], owner[b]), max(owner[a], owner[b])))
    return out


@pytest.mark.parametrize("per", [1, 0])
def test_delaunay_links_equal_the_continuum_triangulation(oracle_mod, per):
    """On a jittered triangular arrangement (no four centres near a common circle, Voronoi edges many lattice
    units long) the links read off the digital Voronoi vertices are exactly the continuum Delaunay links."""
    nx, ny, cols, rows = 120, 104, 6, 6
    pts = _triangular_arrangement(nx, ny, cols, rows, jitter=3.0, seed=11 + per)
    col = oracle_mod.voronoi(nx, ny, per, pts)
    links, n = oracle_mod.delaunay(col, per)
    got = set(map(tuple, links.tolist()))
    assert n == len(links) == len(got)
    assert links.tolist() == [list(p) for p in sorted(got)]   # lexicographic order, a < b
    assert got == _continuum_links(pts, nx, ny, per)
    if per:
        assert n == 3 * cols * rows                     # Euler: a triangulation of the torus has 3 V edges
        deg = np.bincount(links.ravel(), minlength=cols * rows)
        assert (deg == 6).all()


def test_delaunay_two_droplets_between_walls(oracle_mod):
    """Two cells separated by one edge running from wall to wall: the edge ends in no three-cell vertex, the wall
    colour of R24 makes its ends vertices; without walls (y periodic) the ring of two cells has no vertex at all."""
    nx, ny = 32, 12
    c = [[8.0, 6.0], [24.0, 6.0]]
    links, n = oracle_mod.delaunay(oracle_mod.voronoi(nx, ny, 0, c), 0)
    assert links.tolist() == [[0, 1]] and n == 1
    links, n = oracle_mod.delaunay(oracle_mod.voronoi(nx, ny, 1, c), 1)
    assert n == 0


def test_delaunay_four_colour_vertex_takes_the_main_diagonal(oracle_mod):
    """Four quadrant cells on a doubly periodic lattice meet in 2 x 2 blocks of four colours: sides + the pair
    on the block's main diagonal (x, y)-(x+1, y+1) (R24); the anti-diagonal pair is not linked by such a block."""
    nx = ny = 8
    col = np.zeros((ny, nx), np.int32)
    col[:4, 4:] = 1
    col[4:, :4] = 2
    col[4:, 4:] = 3
    links, _ = oracle_mod.delaunay(col, 1)
    # blocks: at (3,3): [[0,1],[2,3]] -> main 0-3; at (7,3): [[1,0],[3,2]] -> main 1-2; (3,7): [[2,3],[0,1]] -> 2-1;
    # (7,7): [[3,2],[1,0]] -> 3-0: both diagonals appear through DIFFERENT vertices of the torus
    assert links.tolist() == [[0, 1], [0, 2], [0, 3], [1, 2], [1, 3], [2, 3]]
    # between walls only the vertices at (3,3) and (7,3) exist, plus the wall vertices linking 0-1 and 2-3
    links, _ = oracle_mod.delaunay(col, 0)
    assert links.tolist() == [[0, 1], [0, 2], [0, 3], [1, 2], [1, 3], [2, 3]]
    # a single four-colour block, no seam (a 2 x 2 lattice between walls): sides + the main diagonal only
    links, _ = oracle_mod.delaunay(np.array([[0, 1], [2, 3]], np.int32)[:, [0, 1]], 0)
    assert [1, 2] in links.tolist() and [0, 3] in links.tolist()  # x periodic: block (1, 0) is [[1, 0], [3, 2]]


def test_delaunay_max_links_truncates_but_counts(oracle_mod):
    nx, ny = 60, 52
    pts = _triangular_arrangement(nx, ny, 3, 4, jitter=1.0, seed=3)
    col = oracle_mod.voronoi(nx, ny, 1, pts)
    full, n = oracle_mod.delaunay(col, 1)
    part, m = oracle_mod.delaunay(col, 1, max_links=5)
    assert m == n == 36 and len(part) == 5 and part.tolist() == full[:5].tolist()


# ---------------------------------------------------------------- R25: matching and T1 events

def test_match_follows_small_displacements(oracle_mod):
    nx, ny = 120, 104
    pts = _triangular_arrangement(nx, ny, 6, 6, jitter=3.0, seed=21)
    col = oracle_mod.voronoi(nx, ny, 0, pts)
    rng = np.random.default_rng(2)
    perm = rng.permutation(len(pts))
    moved = pts[perm] + (rng.random(pts.shape) - 0.5) * 4.0
    moved[:, 0] %= nx
    assert (oracle_mod.match(col, 0, moved) == perm).all()


def test_displacements_minimum_image(oracle_mod):
    """d_i = X_i(now) - X_map[i](past): through the periodic seam in x always, in y only when periodic; (0, 0) unmatched."""
    nx, ny = 100, 40
    past = np.array([[98.0, 5.0], [10.0, 38.5], [50.0, 20.0]])
    now = np.array([[50.5, 19.0], [1.5, 6.0], [12.0, 1.0], [70.0, 7.0]])
    mp = np.array([2, 0, 1, -1], dtype=np.int32)
    d = oracle_mod.displacements(nx, ny, 0, past, now, mp)
    assert np.allclose(d, [[0.5, -1.0], [3.5, 1.0], [2.0, -37.5], [0.0, 0.0]], rtol=0, atol=1e-15)
    d = oracle_mod.displacements(nx, ny, 1, past, now, mp)
    assert np.allclose(d, [[0.5, -1.0], [3.5, 1.0], [2.0, 2.5], [0.0, 0.0]], rtol=0, atol=1e-15)


def _grid_triangulation(cols, rows):
    """Links of a cols x rows grid of points, every square cut by its (i, j)-(i+1, j+1) diagonal."""
    idx = lambda i, j: j * cols + i
    L = set()
    for j in range(rows):
        for i in range(cols):
            if i + 1 < cols:
                L.add((idx(i, j), idx(i + 1, j)))
            if j + 1 < rows:
                L.add((idx(i, j), idx(i, j + 1)))
            if i + 1 < cols and j + 1 < rows:
                L.add((idx(i, j), idx(i + 1, j + 1)))
    return L, idx


def test_t1_hand_made_flip(oracle_mod):
    """The paper's Fig. 2(b): quadrilateral a, b, c, d; the diagonal a-b is replaced by c-d."""
    a, b, c, d = 0, 3, 1, 2
    sides = [(0, 1), (0, 2), (1, 3), (2, 3)]
    past = sorted(sides + [(a, b)])
    now = sorted(sides + [(c, d)])
    ev, n = oracle_mod.t1_events(past, now)
    assert n == 1 and ev.tolist() == [[0, 3, 1, 2]]
    assert oracle_mod.t1_events(past, past)[1] == 0
    assert oracle_mod.t1_events(past, sorted(sides))[1] == 0           # a link lost, none gained: not a T1
    assert oracle_mod.t1_events(sorted(sides), now)[1] == 0            # a link gained, none lost
    assert oracle_mod.t1_events(past, sorted(sides[1:] + [(c, d)]))[1] == 0  # the quadrilateral did not survive
    # the present frame numbers its droplets differently: map[now index] = past index
    perm = np.array([2, 0, 3, 1], dtype=np.int32)   # now droplet k is past droplet perm[k]
    inv = np.argsort(perm)
    now_renum = [(int(inv[p]), int(inv[q])) for p, q in now]
    ev, n = oracle_mod.t1_events(past, now_renum, perm)
    assert n == 1 and ev.tolist() == [[0, 3, 1, 2]]
    # an unmatched droplet (-1) removes its links: the quadrilateral is incomplete, no event
    perm2 = perm.copy()
    perm2[inv[1]] = -1
    assert oracle_mod.t1_events(past, now_renum, perm2)[1] == 0


def test_t1_flips_of_a_triangulated_grid(oracle_mod):
    """Flip the diagonals of several non-adjacent squares of a triangulated grid: exactly those flips come back,
    in lexicographic order."""
    cols, rows = 7, 6
    L, idx = _grid_triangulation(cols, rows)
    flips = [(0, 0), (2, 1), (4, 3), (5, 0), (1, 4)]
    now = set(L)
    expect = []
    for i, j in flips:
        a, b = idx(i, j), idx(i + 1, j + 1)
        c, d = idx(i + 1, j), idx(i, j + 1)
        now.remove((a, b))
        now.add((min(c, d), max(c, d)))
        expect.append([a, b, min(c, d), max(c, d)])
    ev, n = oracle_mod.t1_events(sorted(L), sorted(now))
    assert n == len(flips) and ev.tolist() == sorted(expect)


# ---------------------------------------------------------------- R26: droplet Nusselt number, Eq. (25)

@pytest.mark.parametrize("tau_g", [0.8, 1.0, 1.3])
def test_droplet_nusselt_closed_form(oracle_mod, tau_g):
    """Uniform rise U through the linear conduction profile between walls: at a droplet whose centre is nearest
    to row y_i, u_y T - kappa d_y T = U T(y_i) + kappa dT / ny, so Nu_i = 1 + U T(y_i) ny / (kappa dT) (Eq. (25)
    with Eq. (20)); rows next to a wall use the wall temperature in the face value (R10) and give the same."""
    nx, ny, U, Tb, Tt = 24, 16, 0.011, 0.9, 0.1
    o = oracle_mod.Oracle(nx, ny, tau=1.0, tau_g=tau_g, T_bottom=Tb, T_top=Tt)
    Trow = Tb + (Tt - Tb) * (np.arange(ny) + 0.5) / ny
    Tl = Trow[:, None].repeat(nx, 1)
    f = _linear_pops(np.full((ny, nx), 0.5), 0.0, U)
    o.set_populations(f, 1.4 * f, _linear_pops(Tl, 0.0, 0.0))
    centres = np.array([[3.2, 0.4], [10.6, 7.49], [23.7, 15.2], [5.0, 8.5], [0.49, 3.0]])
    rows = np.array([0, 7, 15, 9, 3])   # floor(c_y + 1/2)
    kappa, dT = (tau_g - 0.5) / 3, Tb - Tt
    expect = 1 + U * Trow[rows] * ny / (kappa * dT)
    assert np.allclose(o.droplet_nusselt(centres), expect, rtol=1e-12, atol=0)


def test_droplet_nusselt_reads_the_nearest_site(oracle_mod):
    """A non-uniform state: Nu_i equals the Eq. (24) integrand of the site floor(X_i + 1/2) (x wrapped)."""
    nx, ny = 12, 10
    rng = np.random.default_rng(8)
    o = oracle_mod.Oracle(nx, ny, tau=1.0, tau_g=0.9, T_bottom=1.0, T_top=0.0)
    T = 0.2 + 0.6 * rng.random((ny, nx))
    uy = 0.02 * (rng.random((ny, nx)) - 0.5)
    f = _linear_pops(np.full((ny, nx), 0.5), 0.0, uy)
    o.set_populations(f, f, _linear_pops(T, 0.0, 0.0))
    centres = np.array([[11.6, 4.4], [3.3, 5.7]])   # -> sites (0, 4) and (3, 6)
    kappa = (0.9 - 0.5) / 3
    exp = []
    for x, y in ((0, 4), (3, 6)):
        dyT = 0.5 * (T[y + 1, x] + T[y, x]) - 0.5 * (T[y, x] + T[y - 1, x])
        exp.append((uy[y, x] * T[y, x] - kappa * dyT) / (kappa * 1.0 / ny))
    assert np.allclose(o.droplet_nusselt(centres), exp, rtol=1e-12, atol=1e-15)


def test_voronoi_at_is_voronoi_on_listed_sites(oracle_mod):
    rng = np.random.default_rng(4)
    nx, ny = 50, 31
    c = rng.random((9, 2)) * [nx, ny]
    full = oracle_mod.voronoi(nx, ny, 0, c)
    sites = rng.integers(0, nx * ny, 200)
    assert (oracle_mod.voronoi_at(nx, ny, 0, c, sites) == full.ravel()[sites]).all()


# ---------------------------------------------------------------- R27: trapezoidal rough walls; R29: perturbation

def test_rough_walls_rectangles_are_the_post_mask(oracle_mod):
    """alpha = 0: "a simple rectangular-shape roughness" (L366) = the structured posts of the headline config."""
    import inputs
    for nx, ny, w, h, lam in ((64, 24, 4, 4, 16), (150, 40, 10, 7, 30), (33, 12, 5, 3, 11)):
        assert (oracle_mod.rough_walls(nx, ny, 1, 1, w, h, lam, 0.0, 0) == inputs.post_mask(nx, ny, w, h, lam)).all()
        only_down = oracle_mod.rough_walls(nx, ny, 0, 1, w, h, lam, 0.0, 1)
        assert only_down[ny // 2:].sum() == 0 and (only_down[:h] == inputs.post_mask(nx, ny, w, h, lam)[:h]).all()


@pytest.mark.parametrize("asym", [0, 1])
def test_rough_walls_trapezoid_shape(oracle_mod, asym):
    """Table A.6's obstacle: width 10, lambda 150, alpha 0.25 (L446-451).  Row j from the wall loses floor(j tan alpha)
    nodes on the inclined side(s): site counts, the vertical side of the asymmetric shape, the mirror symmetry of the
    symmetric one, the top wall as the y-mirror of the bottom wall."""
    nx, ny, w, h, lam, alpha = 300, 60, 10, 9, 150, 0.25
    m = oracle_mod.rough_walls(nx, ny, 1, 1, w, h, lam, alpha, asym)
    cut = [int(np.floor(j * np.tan(alpha))) for j in range(h)]
    assert cut == [0, 0, 0, 0, 1, 1, 1, 1, 2]
    for j in range(h):
        expect = w - cut[j] * (1 if asym else 2)
        assert m[j].sum() == expect * (nx // lam)
        assert (m[j] == m[ny - 1 - j]).all()
        row = m[j, :lam]
        first, last = np.nonzero(row)[0][[0, -1]]
        assert first == (0 if asym else cut[j]) and last == w - 1 - cut[j]
        assert row[first:last + 1].all()                                   # one solid run per obstacle
    assert m[h:ny - h].sum() == 0
    assert (m[:, :lam] == m[:, lam:2 * lam]).all()                         # period lambda


def test_velocity_perturbation_closed_form(oracle_mod):
    """R29: densities unchanged, each fluid's momentum grows by rho_l du, so on a rest state without forces
    u^(H) = du = (0, A sin(2 pi x / nx) sin(pi (y + 1/2) / ny)); solid sites untouched; A = 0 is a no-op."""
    nx, ny, A = 24, 16, 1e-3
    rng = np.random.default_rng(0)
    rA, rB = 0.5 + rng.random((ny, nx)), 0.2 + rng.random((ny, nx))
    solid = np.zeros((ny, nx), np.uint8)
    solid[:2, 3:6] = 1
    o = oracle_mod.Oracle(nx, ny, tau=1.0, thermal=0)
    o.set_solid(solid)
    o.set_fields(rA, rB, np.zeros((ny, nx)))
    f0 = [p.copy() for p in o.get_populations()]
    o.perturb_velocity(0.0)
    assert all((p == q).all() for p, q in zip(o.get_populations(), f0))
    o.perturb_velocity(A)
    fA, fB, g = o.get_populations()
    fl = solid == 0
    assert (g == f0[2]).all() and (fA[:, ~fl] == f0[0][:, ~fl]).all()
    assert np.abs(fA.sum(0) - f0[0].sum(0)).max() < 2e-16 * 4 and np.abs(fB.sum(0) - f0[1].sum(0)).max() < 2e-16 * 4
    du = A * np.sin(2 * np.pi * np.arange(nx) / nx)[None, :] * np.sin(np.pi * (np.arange(ny) + 0.5) / ny)[:, None]
    jyA, jxA = (fA * _CY).sum(0), (fA * _CX).sum(0)
    assert np.abs(jyA - f0[0].sum(0) * du)[fl].max() < 2e-16 and np.abs(jxA)[fl].max() < 2e-16   # rounding of sums of 9 terms ~ 0.1
    rho_A, rho_B, u, T = o.fields()
    assert np.abs(u[1] - du)[fl].max() < 3e-16 and np.abs(u[0])[fl].max() < 3e-16 and np.abs(du).max() > 0.9 * A


def test_honeycomb_centres_arrangement():
    """L266: honeycomb structure of ndx x ndy droplets: equal spacing along x, rows offset by half a spacing."""
    import inputs
    nx, ny, ndx, ndy = 120, 104, 6, 6
    c = inputs.honeycomb_centres(nx, ny, ndx, ndy)
    assert c.shape == (36, 2)
    rows = c.reshape(ndy, ndx, 2)
    assert np.allclose(np.diff(rows[:, :, 0], axis=1), nx / ndx) and np.allclose(rows[1, :, 0] - rows[0, :, 0], nx / ndx / 2)
    assert np.allclose(np.diff(rows[:, 0, 1]), ny / ndy) and rows[0, 0, 1] == ny / ndy / 2
    cp = inputs.honeycomb_centres(nx, ny, ndx, ndy, post_h=4)
    assert cp[:, 1].min() == 4 + (ny - 8) / ndy / 2 and np.isclose(cp[:, 1].max(), ny - 4 - (ny - 8) / ndy / 2)
