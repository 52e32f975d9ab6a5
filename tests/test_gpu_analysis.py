"""GPU parity of the droplet analysis, second stage (tlb_voronoi, tlb_delaunay, tlb_droplet_match, tlb_t1_events,
tlb_droplet_nusselt; PAPER section 2.4, Eq. (25); readings R23-R26) against the oracle's brute force on
the same seeded inputs.  Integer outputs must be bit-identical."""
import numpy as np
import pytest

import inputs
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tlbmod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2109_12565_b200 import binding
    binding.load_library()
    return binding


def _np(t):
    return t.cpu().numpy()


def _dev(tlb, a, dtype=None):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype, device=tlb.device)


def _centres(kind, nx, ny, n, seed):
    """Seeded centre sets: 'rsa' = the input recipe's random sequential addition, 'random' = uniform (cells of very
    different sizes), 'lattice' = integer / half-integer coordinates (many exactly equidistant sites)."""
    if kind == "rsa":
        r = max(2.0, 0.25 * np.sqrt(nx * ny / max(n, 1)))
        return np.array(inputs.place_droplets(nx, ny, seed, n, r, 2.0)).reshape(-1, 2)
    k = np.arange(n)
    if kind == "random":
        return np.stack([inputs.uniform(seed, 5, 2 * k) * nx, inputs.uniform(seed, 5, 2 * k + 1) * ny], 1)
    c = np.stack([np.floor(inputs.uniform(seed, 6, 2 * k) * 2 * nx) / 2, np.floor(inputs.uniform(seed, 6, 2 * k + 1) * 2 * ny) / 2], 1)
    return np.unique(c, axis=0)


CASES = [("rsa", 128, 64, 12, 0), ("rsa", 250, 137, 60, 0), ("random", 257, 131, 40, 1), ("random", 200, 46, 150, 0),
         ("lattice", 96, 80, 70, 1), ("lattice", 64, 48, 30, 0), ("random", 7, 5, 2, 0), ("random", 33, 9, 1, 1),
         ("rsa", 512, 256, 110, 0)]


@pytest.mark.parametrize("kind,nx,ny,n,per", CASES)
def test_voronoi_and_delaunay_bit_exact(tlbmod, oracle_mod, kind, nx, ny, n, per):
    import torch
    c = _centres(kind, nx, ny, n, 3)
    n = len(c)
    t = tlbmod.TLB(nx, ny, periodic_y=per)
    col = t.voronoi(_dev(t, c, torch.float64))
    ocol = oracle_mod.voronoi(nx, ny, per, c)
    assert (_np(col) == ocol).all()
    links, nl = t.delaunay(col, n)
    olinks, onl = oracle_mod.delaunay(ocol, per)
    assert nl == onl and (_np(links) == olinks).all()
    # truncated output: the count is still the full one, the prefix is the same
    if onl > 3:
        part, nl2 = t.delaunay(col, n, max_links=3)
        assert nl2 == onl and (_np(part) == olinks[:3]).all()


def test_voronoi_no_centres_and_errors(tlbmod):
    import torch
    t = tlbmod.TLB(32, 16)
    col = t.voronoi(torch.zeros((0, 2), dtype=torch.float64, device=t.device))
    assert (_np(col) == -1).all()
    links, nl = t.delaunay(col, 0)
    assert nl == 0
    with pytest.raises(tlbmod.TLBError):
        t.voronoi(torch.zeros((32 * 16, 2), dtype=torch.float64, device=t.device))  # n > nx ny / 4


def test_config3_size_voronoi_delaunay(tlbmod, oracle_mod):
    """2048 x 1024 with the 1000 centres of BASELINE config 3's input recipe: whole colouring and link list."""
    import torch
    cfg = inputs.config(3)
    nx, ny, ini = cfg["nx"], cfg["ny"], cfg["init"]
    c = np.array(inputs.place_droplets(nx, ny, cfg["seed"], ini["n_droplets"], ini["droplet_radius"], ini["min_gap"])).reshape(-1, 2)
    t = tlbmod.TLB(nx, ny)
    col = t.voronoi(_dev(t, c, torch.float64))
    ocol = oracle_mod.voronoi(nx, ny, 0, c)
    assert (_np(col) == ocol).all()
    links, nl = t.delaunay(col, len(c))
    olinks, onl = oracle_mod.delaunay(ocol, 0)
    assert nl == onl and (_np(links) == olinks).all()
    assert 2.5 * len(c) < nl < 3 * len(c)   # a planar triangulation with a boundary


def test_config4_size_sampled(tlbmod, oracle_mod):
    """4096 x 2048, the 4000 centres of the headline config: colours on 20 000 sampled sites (plus the sites around
    200 Voronoi vertices, where the decision is closest) against the oracle; the links against what a triangulation
    of the strip must satisfy."""
    import torch
    cfg = inputs.config(4)
    nx, ny, ini = cfg["nx"], cfg["ny"], cfg["init"]
    c = np.array(inputs.place_droplets(nx, ny, cfg["seed"], ini["n_droplets"], ini["droplet_radius"], ini["min_gap"],
                                       post_h=cfg["posts"][1])).reshape(-1, 2)
    n = len(c)
    t = tlbmod.TLB(nx, ny)
    col = t.voronoi(_dev(t, c, torch.float64))
    links, nl = t.delaunay(col, n)
    colh = _np(col)
    sites = (inputs.uniform(77, 3, np.arange(20000)) * nx * ny).astype(np.int64)
    # sites in 2 x 2 blocks with three colours
    blk = (colh[:-1, :-1] != colh[1:, 1:]) & (colh[:-1, 1:] != colh[1:, :-1]) & (colh[:-1, :-1] != colh[:-1, 1:])
    vy, vx = np.nonzero(blk)
    pick = np.arange(0, len(vy), max(1, len(vy) // 200))
    near = np.concatenate([(vy[pick] + dy) * nx + vx[pick] + dx for dy in (0, 1) for dx in (0, 1)])
    sites = np.concatenate([sites, near])
    assert (colh.ravel()[sites] == oracle_mod.voronoi_at(nx, ny, 0, c, sites)).all()
    L = _np(links)
    assert nl == len(L) and (L[:, 0] < L[:, 1]).all()
    key = L[:, 0].astype(np.int64) * n + L[:, 1]
    assert (np.diff(key) > 0).all()                          # sorted, distinct
    deg = np.bincount(L.ravel(), minlength=n)
    assert deg.min() >= 2 and 2.5 * n < nl <= 3 * n - 3      # planar: E <= 3 V - 3; almost all faces are triangles
    # every link joins two droplets whose cells touch: their centres are closer than the two largest cell diameters
    d = c[L[:, 0]] - c[L[:, 1]]
    d[:, 0] -= nx * np.round(d[:, 0] / nx)
    assert np.hypot(d[:, 0], d[:, 1]).max() < 6 * np.sqrt(nx * ny / n)


def _sheared_grid(nx, ny, cols, rows, shear, seed):
    """A slightly irregular square arrangement: the sign of `shear` decides which diagonal of every square is the
    Delaunay link, so going from +shear to -shear flips the diagonals (T1 events)."""
    ax, ay = nx / cols, ny / rows
    k = np.arange(cols * rows)
    i, j = k % cols, k // cols
    jit = (np.stack([inputs.uniform(seed, 7, 2 * k), inputs.uniform(seed, 7, 2 * k + 1)], 1) - 0.5) * 0.02 * ax
    c = np.stack([(i + 0.5) * ax + shear * ax * (j - rows / 2), (j + 0.5) * ay], 1) + jit
    c[:, 0] %= nx
    return c


@pytest.mark.parametrize("per", [0, 1])
def test_t1_events_between_two_frames(tlbmod, oracle_mod, per):
    """Two frames of a sheared square arrangement through the whole chain (voronoi -> delaunay -> match -> T1) on both
    sides; the present frame lists its droplets in another order."""
    import torch
    nx, ny, cols, rows = 240, 192, 10, 8
    past = _sheared_grid(nx, ny, cols, rows, +0.06, 1)
    perm = np.argsort(inputs.uniform(5, 8, np.arange(cols * rows)))
    now = _sheared_grid(nx, ny, cols, rows, -0.06, 1)[perm]
    t = tlbmod.TLB(nx, ny, periodic_y=per)
    cp, cn = t.voronoi(_dev(t, past, torch.float64)), t.voronoi(_dev(t, now, torch.float64))
    lp, nlp = t.delaunay(cp, len(past))
    ln, nln = t.delaunay(cn, len(now))
    mp = t.droplet_match(cp, _dev(t, now, torch.float64))
    ev, ne = t.t1_events(lp, ln, len(past), mp)
    ocp, ocn = oracle_mod.voronoi(nx, ny, per, past), oracle_mod.voronoi(nx, ny, per, now)
    olp, oln = oracle_mod.delaunay(ocp, per)[0], oracle_mod.delaunay(ocn, per)[0]
    omp = oracle_mod.match(ocp, per, now)
    oev, one = oracle_mod.t1_events(olp, oln, omp)
    assert (omp == perm).all() and (_np(mp) == omp).all()
    assert (_np(lp) == olp).all() and (_np(ln) == oln).all()
    assert ne == one and (_np(ev) == oev).all()
    assert one >= (cols - 1) * (rows - 3)   # the interior squares all flip
    disp = t.droplet_displacements(_dev(t, past, torch.float64), _dev(t, now, torch.float64), mp)
    odisp = oracle_mod.displacements(nx, ny, per, past, now, omp)
    assert (_np(disp) == odisp).all() and np.abs(odisp[:, 0]).max() > 1.0
    # truncation keeps the count and the sorted prefix
    ev2, ne2 = t.t1_events(lp, ln, len(past), mp, max_events=5)
    assert ne2 == one and (_np(ev2) == oev[:5]).all()
    # no rearrangement between a frame and itself
    assert t.t1_events(lp, lp, len(past))[1] == 0


def test_t1_events_on_link_lists(tlbmod, oracle_mod):
    """Hand-made link lists (a triangulated grid with some diagonals flipped, droplets renumbered, one unmatched)."""
    import torch
    cols, rows = 9, 7
    idx = lambda i, j: j * cols + i
    L = set()
    for j in range(rows):
        for i in range(cols):
            if i + 1 < cols: L.add((idx(i, j), idx(i + 1, j)))
            if j + 1 < rows: L.add((idx(i, j), idx(i, j + 1)))
            if i + 1 < cols and j + 1 < rows: L.add((idx(i, j), idx(i + 1, j + 1)))
    now = set(L)
    for i, j in [(0, 0), (2, 1), (4, 3), (6, 5), (7, 0), (1, 4)]:
        now.remove((idx(i, j), idx(i + 1, j + 1)))
        now.add(tuple(sorted((idx(i + 1, j), idx(i, j + 1)))))
    n = cols * rows
    perm = np.argsort(inputs.uniform(2, 9, np.arange(n))).astype(np.int32)   # now droplet k is past droplet perm[k]
    inv = np.argsort(perm)
    now_r = np.array(sorted(tuple(sorted((inv[a], inv[b]))) for a, b in now), dtype=np.int32)
    past = np.array(sorted(L), dtype=np.int32)
    mp = perm.copy()
    mp[inv[idx(5, 4)]] = -1   # one droplet of the (4, 3) square lost: that flip must not be reported
    t = tlbmod.TLB(64, 32)
    ev, ne = t.t1_events(_dev(t, past), _dev(t, now_r), n, _dev(t, mp))
    oev, one = oracle_mod.t1_events(past, now_r, mp)
    assert ne == one == 5 and (_np(ev) == oev).all()


def test_droplet_nusselt_parity(tlbmod, oracle_mod):
    """Config 1 (paper physics, posts) after 300 steps: centres from the droplet labelling, Nu_i of Eq. (25)."""
    cfg = dict(inputs.config(1, physics="paper"), posts=(4, 4, 16))
    nx, ny = cfg["nx"], cfg["ny"]
    solid, rA, rB, T = inputs.make_config_inputs(cfg)
    t = tlbmod.TLB(nx, ny, params=tlbmod.params_from_config(cfg))
    t.set_solid(solid)
    t.set_fields(rA, rB, T)
    o = oracle_mod.Oracle(nx, ny, **cfg["params"])
    o.set_solid(solid)
    o.set_fields(rA, rB, T)
    t.step(300)
    o.step(300)
    B_th = 0.5 * (cfg["init"]["rho_in"] + cfg["init"]["rho_out"])
    _, k, stats = t.droplets(B_th, 64)
    _, ok, ostats = o.droplets(B_th, 64)
    assert k == ok and k >= 8 and (_np(stats) == ostats).all()
    nu = _np(t.droplet_nusselt(stats[:, 2:4]))
    onu = o.droplet_nusselt(ostats[:, 2:4])
    assert np.abs(nu - onu).max() <= 1e-12 * max(1.0, np.abs(onu).max())
    assert np.abs(onu).max() > 0.1


def test_delaunay_monitor_files(tlbmod, oracle_mod, tmp_path):
    """The run-time monitor of Table C.12 (monitor.py, reading R32): a honeycomb emulsion checked every 40 steps (time
    sequences, frame files that read back to what the analysis calls return and to the oracle's analysis of the same
    state), then two hand-made frames of a sheared arrangement whose diagonals flip (events in the trigger directory)."""
    import torch
    from paper_2109_12565_b200 import monitor
    cfg = dict(inputs.config(1, "paper"), nx=192, ny=96)
    cfg["init"] = dict(cfg["init"], droplet_radius=8.0)
    nx, ny = cfg["nx"], cfg["ny"]
    t = tlbmod.TLB(nx, ny, params=tlbmod.params_from_config(cfg))
    t.init_honeycomb(6, 3, 5)
    B_th = 0.5 * (cfg["init"]["rho_in"] + cfg["init"]["rho_out"])
    mon = monitor.DelaunayMonitor(t, B_th, str(tmp_path), max_droplets=64)
    for k in range(3):
        t.step(40)
        ev = mon.check(40 * (k + 1))
        assert len(ev) == 0          # a relaxing honeycomb does not rearrange
    nb = np.loadtxt(tmp_path / "nBubblesOut")
    nl = np.loadtxt(tmp_path / "nLinksOut")
    assert (nb[:, 0] == [40, 80, 120]).all() and (nb[:, 1] == 18).all() and (nl[:, 1] == nl[0, 1]).all() and nl[0, 1] > 30
    cen, links = monitor.read_frame(tmp_path / "delaunayNoTriggerDir" / "delaunayNowTime120")
    fr = mon.frame(120)
    assert (cen == _np(fr.centres)).all() and (links == _np(fr.links)).all()
    # the oracle on the same state (through the populations) finds the same droplets, colouring and links
    o = oracle_mod.Oracle(nx, ny, **cfg["params"])
    o.set_solid(np.zeros((ny, nx), np.uint8))
    o.set_populations(*[_np(p) for p in t.get_populations()])
    _, ok, ostats = o.droplets(B_th, 64)
    assert ok == 18 and (ostats[:, 2:4] == cen).all()
    olinks, _ = oracle_mod.delaunay(oracle_mod.voronoi(nx, ny, 0, ostats[:, 2:4]), 0)
    assert (olinks == links).all()
    # two hand-made frames: every interior diagonal of a sheared square arrangement flips
    NX, NY, cols, rows = 240, 192, 10, 8
    t2 = tlbmod.TLB(NX, NY, periodic_y=1)
    mon2 = monitor.DelaunayMonitor(t2, 0.0, str(tmp_path / "flip"))
    frames = []
    for step, shear in ((10, +0.06), (20, -0.06)):
        c = _dev(t2, _sheared_grid(NX, NY, cols, rows, shear, 1), torch.float64)
        colour = t2.voronoi(c)
        lk, _ = t2.delaunay(colour, len(c))
        frames.append(monitor.Frame(step, len(c), c, colour, lk))
    assert len(mon2.record(frames[0])) == 0
    ev = mon2.record(frames[1])
    oev, one = oracle_mod.t1_events(_np(frames[0].links), _np(frames[1].links), np.arange(cols * rows, dtype=np.int32))
    assert one == len(ev) == 80 and (ev == oev).all()
    brk = np.loadtxt(tmp_path / "flip" / "delaunayTriggerDir" / "breakingLinks", dtype=int)
    ari = np.loadtxt(tmp_path / "flip" / "delaunayTriggerDir" / "arisingLinks", dtype=int)
    assert (brk[:, 0] == 20).all() and (brk[:, 1:] == ev[:, :2]).all() and (ari[:, 1:] == ev[:, 2:]).all()
    pc, pl = monitor.read_frame(tmp_path / "flip" / "delaunayTriggerDir" / "delaunayPastTime20")
    assert (pl == _np(frames[0].links)).all() and (pc == _np(frames[0].centres)).all()
