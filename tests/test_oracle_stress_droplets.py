"""Pins (-m "not gpu") of the oracle's stress field P_xy (reading R21; Eq. (14))
and of its droplet labelling (reading R22; PAPER section 2.4).  Nothing here comes from the CUDA path.

P_xy has no formula in the paper, so it is pinned by what mechanics fixes:
  * single-phase Couette: P_xy = -rho nu (U_t - U_b) / ny exactly, nu = (tau - 1/2)/3 (Eq. (14), Eq. (23));
  * a sheared two-layer fluid (flat interface, forces along y only): the x-averaged stress Pxy_av (L250) is the
    same in every row at steady state, and equal to the momentum the moving walls feed in;
  * -div P = F in its exact lattice form on an arbitrary state at rest (derived in DESIGN.md R21): row sums of the
    interaction part against row sums of the force, row by row when the interactions reach one row
    (nearest-neighbour couplings) and in the first moment for all couplings, plus the momentum one step moves.
"""
import numpy as np
import pytest

import inputs
CX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1])[:, None, None]
CY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1])[:, None, None]
WQ = np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)[:, None, None]


@pytest.mark.parametrize("tau", [0.8, 1.0, 1.4])
def test_stress_single_phase_couette(oracle_mod, tau):
    nx, ny, Ub, Ut = 6, 16, -0.01, 0.03
    o = oracle_mod.Oracle(nx, ny, tau=tau, thermal=0, u_wall_bottom=Ub, u_wall_top=Ut)
    f = np.full((ny, nx), 0.5)
    o.set_fields(f, 1.4 * f, 0 * f)
    nu = (tau - 0.5) / 3.0
    o.step(int(40 * ny * ny / nu / 10))
    rho = o.fields()[0] + o.fields()[1]
    expect = -rho * nu * (Ut - Ub) / ny
    P = o.stress_xy()
    assert np.abs(P / expect - 1).max() < 1e-8, np.abs(P / expect - 1).max()
    assert np.abs(o.x_average_stress() / expect.mean(axis=1) - 1).max() < 1e-8


def test_stress_sign_and_transpose(oracle_mod):
    """A uniform stream (U_x, U_y) at equilibrium carries P_xy = rho U_x U_y (the advective momentum flux): fixes
    the sign, the c_x c_y pairing of the diagonal directions and the 1/2 (f + f*) average (f* = f here)."""
    nx, ny, Ux, Uy = 8, 6, 0.03, -0.02
    o = oracle_mod.Oracle(nx, ny, tau=0.9, thermal=0, periodic_y=1)
    rho = np.full((ny, nx), 0.8)
    cu = CX * Ux + CY * Uy
    feq = WQ * rho * (1 + 3 * cu + 4.5 * cu * cu - 1.5 * (Ux * Ux + Uy * Uy))
    o.set_populations(0.25 * feq, 0.75 * feq, 0 * feq)
    assert np.abs(o.stress_xy() - 0.8 * Ux * Uy).max() < 1e-16


def test_stress_two_layer_couette_is_uniform(oracle_mod):
    """Two immiscible layers (A-rich below, B-rich above) sheared between moving walls: at steady state the
    x-averaged total stress is the same in every row, interface included, although density, forces and the
    velocity gradient all change across it."""
    nx, ny, Ub, Ut = 4, 48, -0.02, 0.02
    par = dict(inputs.PAPER_PHYSICS, thermal=0, alpha_g=0.0, u_wall_bottom=Ub, u_wall_top=Ut, tau=1.0)
    o = oracle_mod.Oracle(nx, ny, **par)
    lower = (np.arange(ny) < ny // 2)[:, None].repeat(nx, 1)
    o.set_fields(np.where(lower, 1.36, 0.155), np.where(lower, 0.155, 1.36), np.zeros((ny, nx)))
    o.step(60000)
    av = o.x_average_stress()
    rho = (o.fields()[0] + o.fields()[1]).mean(axis=1)
    assert rho.max() / rho.min() > 1.05  # the layers are there
    assert av.max() < 0 and (av.max() - av.min()) < 1e-7 * abs(av.mean()), (av.min(), av.max())  # residual: the interface still creeps
    # and it is the viscous stress of the bulk of either layer: -rho nu du/dy
    u = o.x_average()
    k = ny // 4
    assert abs(av[k] / (-rho[k] * (1.0 - 0.5) / 3.0 * (u[k + 1] - u[k - 1]) / 2) - 1) < 1e-6


def _blob_densities(nx, ny, seed):
    """Two density fields that are uniform near the walls and busy in the middle (state at rest, R14)."""
    x = np.arange(nx)[None, :] * (2 * np.pi / nx)
    y = np.arange(ny)[:, None]
    env = np.exp(-((y - 0.5 * ny) / (0.12 * ny)) ** 4)
    env[np.abs(y[:, 0] - 0.5 * ny) > 0.38 * ny] = 0.0
    ph = inputs.uniform(seed, 11, np.arange(6)) * 2 * np.pi
    rA = 0.7 + env * (0.35 * np.sin(x + ph[0]) * np.cos(0.4 * y + ph[1]) + 0.2 * np.cos(3 * x + ph[2]))
    rB = 0.6 + env * (0.3 * np.cos(2 * x + ph[3]) * np.sin(0.3 * y + ph[4]) - 0.15 * np.sin(x + ph[5]))
    return rA, rB


@pytest.mark.parametrize("couplings", ["nn_only", "all"])
@pytest.mark.parametrize("tau", [0.8, 1.0])
def test_stress_interaction_part_balances_the_forces(oracle_mod, couplings, tau):
    """-div P = F in its exact lattice form.  State at rest (f = w rho): the arriving populations carry no P_xy,
    the leaving ones sum_i c_ix c_iy f*_l,i = tau F_l,x F_l,y / rho_l (Eqs. (2), (3), (6) with u = 0), so the kinetic
    part is K = 1/2 tau sum_l F_l,x F_l,y / rho_l and I = P_xy - K is the interaction part.  Every pair interaction
    (x, x + c) hands its x-force across the c_y planes between its sites, and the tensor gives half of it to each
    end, hence with Ibar(y), Fbar(y) the row sums of I and of F_x = F_A,x + F_B,x:
        sum_y Ibar(y) = sum_y y Fbar(y)                               (all couplings)
        Ibar(y + 1) - Ibar(y) = -1/2 [Fbar(y + 1) + Fbar(y)]           (couplings that reach one row)
    and one time step moves the momentum M(y) of the rows by sum_y y dM(y) = sum (2 K + I)."""
    nx, ny = 20, 44
    par = dict(inputs.PAPER_PHYSICS, thermal=0, alpha_g=0.0, tau=tau)
    if couplings == "nn_only":
        par.update(G11r=0.0, G22r=0.0, G11a=-1.3, G22a=-1.1)  # the p-weighted family reaches two rows: off
    o = oracle_mod.Oracle(nx, ny, **par)
    rA, rB = _blob_densities(nx, ny, 5)
    o.set_fields(rA, rB, 0 * rA)
    P = o.stress_xy()
    FA, FB = o.forces()
    K = 0.5 * tau * (FA[0] * FA[1] / rA + FB[0] * FB[1] / rB)
    Ibar = (P - K).sum(axis=1)
    Fbar = (FA[0] + FB[0]).sum(axis=1)
    assert np.abs(Fbar).max() > 1e-4 and np.abs(Ibar).max() > 1e-4  # a busy state, not a trivial one
    yy = np.arange(ny)
    assert abs(Ibar.sum() - (yy * Fbar).sum()) < 1e-14 * ny * nx, (Ibar.sum(), (yy * Fbar).sum())
    if couplings == "nn_only":
        assert np.abs((Ibar[1:] - Ibar[:-1]) + 0.5 * (Fbar[1:] + Fbar[:-1])).max() < 1e-14 * nx
    M0 = o.row_momentum_x()
    o.step(1)
    dM = o.row_momentum_x() - M0
    assert abs((yy * dM).sum() - (2 * K.sum() + Ibar.sum())) < 1e-14 * ny * nx


def test_stress_is_zero_on_solid_sites_and_uses_wall_values(oracle_mod):
    """Posts: P_xy = 0 on solid sites; a fluid site next to a post corner sees the wall pseudopotential in the
    interaction part (L155): for a uniform fluid at rest P_xy(x) = 1/2 sum_c k(c) c_x c_y psi psi(x + c) reduces to
    differences between the wall and the fluid values over the solid neighbours -- evaluated here by hand."""
    nx, ny = 16, 14
    par = dict(inputs.PAPER_PHYSICS, thermal=0, alpha_g=0.0)
    solid = inputs.post_mask(nx, ny, 3, 3, 8)
    o = oracle_mod.Oracle(nx, ny, **par)
    o.set_solid(solid)
    rA0, rB0 = 0.9, 0.3
    o.set_fields(np.full((ny, nx), rA0), np.full((ny, nx), rB0), np.zeros((ny, nx)))
    P = o.stress_xy()
    assert np.all(P[solid == 1] == 0.0)
    w, p = oracle_mod.lattice_weights()
    rho0 = par["rho0"]
    pss = lambda r: rho0 * (1 - np.exp(-r / rho0))
    full = np.ones((ny + 4, nx), bool)  # rows -2..ny+1: beyond the walls everything is solid
    full[2:-2] = solid == 1
    full[2:-2][solid == 0] = False
    expect = np.zeros((ny, nx))
    for y in range(ny):
        for x in range(nx):
            if solid[y, x]:
                continue
            acc = 0.0
            for dx in range(-2, 3):
                for dy in range(-2, 3):
                    if (dx or dy) and full[y + dy + 2, (x + dx) % nx]:
                        # solid neighbour: wall value instead of the fluid value; the uniform part sums to zero
                        ww, pp = w[(dx, dy)], p[(dx, dy)]
                        acc += dx * dy * (par["G12"] * ww * (rA0 * (par["rho_wall_B"] - rB0) + rB0 * (par["rho_wall_A"] - rA0)) / rho0 ** 2
                                          + (par["G11a"] * ww + par["G11r"] * pp) * pss(rA0) * (pss(par["rho_wall_A"]) - pss(rA0))
                                          + (par["G22a"] * ww + par["G22r"] * pp) * pss(rB0) * (pss(par["rho_wall_B"]) - pss(rB0)))
            expect[y, x] = 0.5 * acc
    assert np.abs(expect).max() > 1e-4
    FA, FB = o.forces()  # the walls push the fluid next to them: kinetic part 1/2 tau sum_l F_l,x F_l,y / rho_l (state at rest)
    expect += np.where(solid == 0, 0.5 * par["tau"] * (FA[0] * FA[1] / rA0 + FB[0] * FB[1] / rB0), 0.0)
    assert np.abs(P - expect).max() < 1e-14


# ---- droplets (section 2.4, R22) -------------------------------------------------------------------------------

def _oracle_with_density(oracle_mod, rhoA, solid=None, periodic_y=0):
    ny, nx = rhoA.shape
    o = oracle_mod.Oracle(nx, ny, thermal=0, periodic_y=periodic_y)
    if solid is not None:
        o.set_solid(solid)
    z = np.zeros((9, ny, nx))
    fA, fB = z.copy(), z.copy()
    fA[0], fB[0] = rhoA, 0.3  # all of the density in the rest population: rho_A = sum_i f_A,i is exactly the input
    o.set_populations(fA, fB, z)
    return o


def test_droplets_hand_made_masks(oracle_mod):
    """Known clusters: a 2x3 block, an L-shape that touches it only diagonally (nearest-neighbour bonds: a separate
    droplet), a single site, a bar that crosses the x seam, a site on a solid node (not bulk)."""
    nx, ny = 12, 8
    m = np.zeros((ny, nx), bool)
    m[1:3, 2:5] = True                      # block: 6 sites, label 1*12+2 = 14
    m[3, 5] = m[4, 5] = m[4, 6] = True      # L: touches the block at (2,4)-(3,5) diagonally only; label 3*12+5 = 41
    m[6, 9] = True                          # single site, label 81
    m[5, [10, 11, 0, 1]] = True             # bar across the seam: label = smallest index = 5*12+0 = 60
    m[0, 7] = True                          # will be made solid
    solid = np.zeros((ny, nx), np.uint8)
    solid[0, 7] = 1
    rhoA = np.where(m, 1.2, 0.1)
    rhoA[2, 3] = 0.6 + 1e-12                # just above the threshold: still bulk
    rhoA[7, 7] = 0.6                        # exactly the threshold: NOT bulk (strict inequality, L198 "larger than")
    o = _oracle_with_density(oracle_mod, rhoA, solid)
    labels, n, st = o.droplets(0.6, 16)
    assert n == 4
    assert labels[0, 7] == -1 and labels[7, 7] == -1
    assert np.array_equal(st[:, 0], [14, 41, 60, 81]) and np.array_equal(st[:, 1], [6, 3, 4, 1])
    assert np.all(labels[1:3, 2:5] == 14) and labels[3, 5] == labels[4, 5] == labels[4, 6] == 41
    assert np.all(labels[5, [10, 11, 0, 1]] == 60) and labels[6, 9] == 81
    assert (labels >= 0).sum() == 14
    assert np.allclose(st[0, 2:], [3.0, 1.5]) and np.allclose(st[1, 2:], [5 + 1 / 3, 3 + 2 / 3])
    # the bar: sites x = 10, 11, 0, 1 -> mean position 11.5 (mod 12), not 5.5
    assert abs(st[2, 2] - 11.5) < 1e-15 and st[2, 3] == 5.0
    assert np.array_equal(st[3, 2:], [9.0, 6.0])
    # truncation: only the first max_droplets rows are written, the count is still complete
    _, n2, st2 = o.droplets(0.6, 2)
    assert n2 == 4 and np.array_equal(st2, st[:2])


def test_droplets_periodic_y_and_walls(oracle_mod):
    nx, ny = 6, 5
    m = np.zeros((ny, nx), bool)
    m[0, 2] = m[4, 2] = True
    rhoA = np.where(m, 1.0, 0.0)
    _, n_w, _ = _oracle_with_density(oracle_mod, rhoA, periodic_y=0).droplets(0.5, 4)
    lab, n_p, st = _oracle_with_density(oracle_mod, rhoA, periodic_y=1).droplets(0.5, 4)
    assert n_w == 2 and n_p == 1
    assert lab[0, 2] == lab[4, 2] == 2 and st[0, 1] == 2 and st[0, 3] == 4.5  # rows 0 and 4 (= -1): centre -0.5 -> 4.5


def test_droplets_discs_centroids_and_shift_invariance(oracle_mod):
    """Seeded discs (the input recipe's droplets): as many clusters as discs, each with the exact lattice-disc
    site count and its centroid within half a site of the disc's centre; shifting the field along x (through the
    seam) shifts centres and keeps counts."""
    nx, ny, r = 96, 64, 6.0
    c = inputs.place_droplets(nx, ny, 3, 9, r, 4.0)
    rA, _, _ = inputs.initial_fields(nx, ny, 3, 9, r, 4.0, 1.0, 0.04, 0.0, 0.0, 0.0)
    o = _oracle_with_density(oracle_mod, rA)
    lab, n, st = o.droplets(0.5, 32)
    assert n == 9
    x = np.arange(nx)[None, :]
    y = np.arange(ny)[:, None]
    for cx, cy in c:
        dx = np.minimum(np.abs(x - cx), nx - np.abs(x - cx))
        inside = dx * dx + (y - cy) ** 2 <= r * r
        k = lab[inside][0]
        assert np.all(lab[inside] == k) and (lab == k).sum() == inside.sum()
        row = st[st[:, 0] == k][0]
        ddx = min(abs(row[2] - cx), nx - abs(row[2] - cx))
        assert row[1] == inside.sum() and ddx < 0.5 and abs(row[3] - cy) < 0.5
    sh = 37
    o2 = _oracle_with_density(oracle_mod, np.roll(rA, sh, axis=1))
    _, n2, st2 = o2.droplets(0.5, 32)
    assert n2 == 9
    a = sorted((round(cnt), round((cx + sh) % nx, 9), round(cy, 9)) for _, cnt, cx, cy in st)
    b = sorted((round(cnt), round(cx % nx, 9), round(cy, 9)) for _, cnt, cx, cy in st2)
    assert a == b


def test_droplets_brute_force_small_random(oracle_mod):
    """Random bulk masks on tiny lattices against a transitive closure of the bond relation written here."""
    for seed in range(6):
        nx, ny = 7, 6
        u = inputs.uniform(seed, 21, np.arange(nx * ny)).reshape(ny, nx)
        bulk = u < 0.55
        per_y = seed % 2
        o = _oracle_with_density(oracle_mod, np.where(bulk, 1.0, 0.0), periodic_y=per_y)
        lab, n, st = o.droplets(0.5, nx * ny // 4)
        comp = {(yy, xx): yy * nx + xx for yy in range(ny) for xx in range(nx) if bulk[yy, xx]}
        changed = True
        while changed:
            changed = False
            for (yy, xx) in comp:
                for dy, dx in ((0, 1), (1, 0)):
                    y2, x2 = yy + dy, (xx + dx) % nx
                    if y2 >= ny:
                        if not per_y:
                            continue
                        y2 = 0
                    if (y2, x2) in comp and comp[(y2, x2)] != comp[(yy, xx)]:
                        lo = min(comp[(y2, x2)], comp[(yy, xx)])
                        comp[(y2, x2)] = comp[(yy, xx)] = lo
                        changed = True
        expect = -np.ones((ny, nx), np.int32)
        for (yy, xx), k in comp.items():
            expect[yy, xx] = k
        assert np.array_equal(lab, expect)
        assert n == len(set(comp.values()))
