"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no moments, forces, collision, streaming):
it only produces the initial density / temperature fields, the solid masks and the parameter
sets of the workloads in BASELINE.json, following the recipe of DESIGN.md ("Input recipe").
Both the oracle and the CUDA path are fed its arrays; `tlb_init(seed)` in the CUDA library
implements the same recipe natively and tests compare the two bit for bit.

The paper's own workloads (prepared honeycomb emulsions, Fig. 3) are not in
the container; these seeded random-sequential-addition emulsions stand in for them.
"""
import numpy as np

_GOLDEN = 0x9E3779B97F4A7C15
_M64 = (1 << 64) - 1


def _mix64(z):
    """SplitMix64 finaliser on uint64 numpy arrays (wrap-around arithmetic)."""
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniform(seed, stream, k):
    """Counter-based uniform in [0,1): top 53 bits of mix64(seed + GOLDEN*(stream*2^40 + k + 1))."""
    k = np.asarray(k, dtype=np.uint64)
    with np.errstate(over="ignore"):
        ctr = np.uint64(stream) * np.uint64(1 << 40) + k + np.uint64(1)
        z = np.uint64(seed & _M64) + np.uint64(_GOLDEN) * ctr
    return (_mix64(z) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


# physics of BASELINE.json's configs ("literal" set) and of the paper's Table A.3 ("paper" set)
LITERAL_PHYSICS = dict(tau=1.0, tau_g=1.0, rho0=1.0, G12=0.405, G11a=-9.0, G11r=8.1, G22a=-9.0, G22r=8.1,
                       rho_wall_A=0.52, rho_wall_B=0.52, T_bottom=1.0, T_top=0.0, T_ref=0.5, alpha_g=1e-4,
                       body_ax=0.0, u_wall_bottom=0.0, u_wall_top=0.0, periodic_y=0, thermal=1)
PAPER_PHYSICS = dict(tau=1.0, tau_g=1.0, rho0=0.83, G12=0.405, G11a=-9.0, G11r=8.1, G22a=-8.0, G22r=7.1,
                     rho_wall_A=0.612, rho_wall_B=0.612, T_bottom=0.5, T_top=-0.5, T_ref=0.0, alpha_g=1.24e-5,
                     body_ax=0.0, u_wall_bottom=0.0, u_wall_top=0.0, periodic_y=0, thermal=1)


def config(index, physics="literal"):
    """Workload `index` (1..5) of BASELINE.json: dict(nx, ny, params, init, steps)."""
    table = {
        1: dict(nx=128, ny=64, n_droplets=12, radius=6.0, seed=1, posts=(0, 0, 0), steps=1000),
        2: dict(nx=512, ny=256, n_droplets=110, radius=10.0, seed=2, posts=(0, 0, 0), steps=20000),
        3: dict(nx=2048, ny=1024, n_droplets=1000, radius=14.0, seed=3, posts=(0, 0, 0), steps=5000),
        4: dict(nx=4096, ny=2048, n_droplets=4000, radius=14.0, seed=4, posts=(4, 4, 16), steps=2000),
        5: dict(nx=8192, ny=4096, n_droplets=16000, radius=14.0, seed=5, posts=(0, 0, 0), steps=1000),
    }
    c = dict(table[index])
    phys = dict(LITERAL_PHYSICS if physics == "literal" else PAPER_PHYSICS)
    if physics == "literal":
        rho_in, rho_out = 1.0, 0.04
    else:
        rho_in, rho_out = 1.36, 0.155
    c["params"] = phys
    c["init"] = dict(n_droplets=c.pop("n_droplets"), droplet_radius=c.pop("radius"), min_gap=4.0,
                     rho_in=rho_in, rho_out=rho_out, noise_amp=1e-3)
    c["name"] = "config%d_%dx%d" % (index, c["nx"], c["ny"])
    return c


def post_mask(nx, ny, post_w, post_h, post_period):
    """Structured rough walls (BASELINE config 4, reading R19): solid iff
    (x mod period) < post_w and (y < post_h or y >= ny - post_h)."""
    m = np.zeros((ny, nx), dtype=np.uint8)
    if post_w > 0 and post_h > 0 and post_period > 0:
        x = np.arange(nx)[None, :]
        y = np.arange(ny)[:, None]
        m[((x % post_period) < post_w) & ((y < post_h) | (y >= ny - post_h))] = 1
    return m


def place_droplets(nx, ny, seed, n_droplets, radius, min_gap, post_h=0):
    """Random sequential addition of equal discs, periodic in x.  Returns an (n, 2) array of
    (cx, cy), or raises if `n_droplets` cannot be placed within 1000*n candidates."""
    r = float(radius)
    y_lo = r + 3.0 + post_h
    y_hi = ny - 1.0 - y_lo
    centres = np.zeros((n_droplets, 2))
    n = 0
    if n_droplets > 0 and y_hi < y_lo:
        raise ValueError("lattice too small for the droplets")
    dmin2 = (2.0 * r + min_gap) * (2.0 * r + min_gap)
    k = 0
    batch = 4096
    while n < n_droplets and k < 1000 * n_droplets:
        ks = np.arange(k, min(k + batch, 1000 * n_droplets), dtype=np.uint64)
        cxs = uniform(seed, 0, 2 * ks) * nx
        cys = y_lo + uniform(seed, 0, 2 * ks + np.uint64(1)) * (y_hi - y_lo)
        for cx, cy in zip(cxs, cys):
            if n:
                dx = np.abs(centres[:n, 0] - cx)
                dx = np.minimum(dx, nx - dx)
                dy = centres[:n, 1] - cy
                if np.any(dx * dx + dy * dy < dmin2):
                    continue
            centres[n] = (cx, cy)
            n += 1
            if n == n_droplets:
                break
        k += batch
    if n < n_droplets:
        raise ValueError("could not place %d droplets" % n_droplets)
    return centres


def honeycomb_centres(nx, ny, ndx, ndy, post_h=0):
    """ndx x ndy centres in a honeycomb (triangular) arrangement between the walls / posts, the paper's own
    initialisation ("droplet initialisation = 1"): row j at y = post_h + (j + 1/2) (ny - 2 post_h) / ndy,
    column i at x = (i + 1/4 + (j mod 2) / 2) nx / ndx."""
    j, i = np.divmod(np.arange(ndx * ndy), ndx)
    ax = float(nx) / float(ndx)
    ay = (float(ny) - 2.0 * float(post_h)) / float(ndy)
    cx = (i.astype(np.float64) + 0.25 + 0.5 * (j % 2).astype(np.float64)) * ax
    cy = float(post_h) + (j.astype(np.float64) + 0.5) * ay
    return np.stack([cx, cy], 1)


def initial_fields(nx, ny, seed, n_droplets, droplet_radius, min_gap, rho_in, rho_out, noise_amp,
                   T_bottom, T_top, solid=None, post_h=0, centres=None):
    """(rho_A, rho_B, T) of the input recipe: droplets rich in A, matrix rich in B, seeded uniform
    noise on fluid sites, linear temperature profile between the walls.  `centres` (n, 2)
    replaces the random sequential addition (e.g. honeycomb_centres)."""
    inside = np.zeros((ny, nx), dtype=bool)
    if centres is not None or n_droplets > 0:
        if centres is None:
            centres = place_droplets(nx, ny, seed, n_droplets, droplet_radius, min_gap, post_h)
        r2 = float(droplet_radius) * float(droplet_radius)
        rr = int(np.ceil(droplet_radius)) + 1
        for cx, cy in centres:
            ys = np.arange(max(0, int(np.floor(cy)) - rr), min(ny, int(np.floor(cy)) + rr + 2))
            xs = np.arange(int(np.floor(cx)) - rr, int(np.floor(cx)) + rr + 2)
            xw = np.mod(xs, nx)
            dx = np.abs(xw.astype(np.float64) - cx)
            dx = np.minimum(dx, nx - dx)
            dy = ys.astype(np.float64) - cy
            hit = (dx * dx)[None, :] + (dy * dy)[:, None] <= r2
            sub = inside[np.ix_(ys, xw)]
            inside[np.ix_(ys, xw)] = sub | hit
    rho_A = np.where(inside, rho_in, rho_out).astype(np.float64)
    rho_B = np.where(inside, rho_out, rho_in).astype(np.float64)
    k = (np.arange(ny, dtype=np.uint64)[:, None] * np.uint64(nx) + np.arange(nx, dtype=np.uint64)[None, :])
    nA = noise_amp * uniform(seed, 1, k)
    nB = noise_amp * uniform(seed, 2, k)
    fluid = np.ones((ny, nx), dtype=bool) if solid is None else (np.asarray(solid) == 0)
    rho_A = np.where(fluid, rho_A + nA, rho_A)
    rho_B = np.where(fluid, rho_B + nB, rho_B)
    yy = np.arange(ny, dtype=np.float64) + 0.5
    Trow = ((T_top - T_bottom) * yy) / ny + T_bottom
    T = np.repeat(Trow[:, None], nx, axis=1)
    return rho_A, rho_B, np.ascontiguousarray(T)


def make_config_inputs(cfg):
    """Everything a run of `cfg` (from config()) needs: solid mask and the three initial fields."""
    nx, ny = cfg["nx"], cfg["ny"]
    pw, ph, pp = cfg["posts"]
    solid = post_mask(nx, ny, pw, ph, pp)
    i, p = cfg["init"], cfg["params"]
    rho_A, rho_B, T = initial_fields(nx, ny, cfg["seed"], i["n_droplets"], i["droplet_radius"], i["min_gap"],
                                     i["rho_in"], i["rho_out"], i["noise_amp"], p["T_bottom"], p["T_top"],
                                     solid=solid, post_h=ph)
    return solid, rho_A, rho_B, T


def smooth_random_fields(nx, ny, seed, T_bottom=1.0, T_top=0.0, amp=0.2):
    """Small generic test input: smooth, strictly positive densities with a few Fourier modes."""
    x = np.arange(nx)[None, :] * (2 * np.pi / nx)
    y = np.arange(ny)[:, None] * (2 * np.pi / max(ny, 1))
    ph = uniform(seed, 7, np.arange(8)) * 2 * np.pi
    rho_A = 0.6 + amp * np.sin(x + ph[0]) * np.cos(y + ph[1]) + 0.5 * amp * np.cos(2 * x + ph[2])
    rho_B = 0.7 + amp * np.cos(x + ph[3]) * np.sin(2 * y + ph[4]) - 0.5 * amp * np.sin(3 * x + ph[5])
    T = 0.5 * (T_bottom + T_top) + 0.3 * (T_bottom - T_top) * np.sin(x + ph[6]) * np.cos(y + ph[7])
    return np.ascontiguousarray(rho_A), np.ascontiguousarray(rho_B), np.ascontiguousarray(T + 0 * rho_A)
