"""ctypes loader for oracle/tlb_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It shares nothing with paper_2109_12565_b200 (the CUDA path) and
neither imports the other.  All arithmetic lives in tlb_oracle.c; this file only marshals
numpy arrays (argument meaning follows PAPER.md Eqs. (1)-(22) and DESIGN.md readings).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tlb_oracle.c")
_LIB = os.path.join(_HERE, "liborc.so")


def build(force=False):
    """Compile the oracle with gcc (-O2, no FMA contraction, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class OrcParams(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in (
        "tau", "tau_g", "rho0", "G12", "G11a", "G11r", "G22a", "G22r", "rho_wall_A", "rho_wall_B",
        "T_bottom", "T_top", "T_ref", "alpha_g", "body_ax", "u_wall_bottom", "u_wall_top")] + [
        ("periodic_y", ctypes.c_int32), ("thermal", ctypes.c_int32)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        lib.orc_create.restype = ctypes.c_void_p
        lib.orc_create.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(OrcParams)]
        lib.orc_destroy.argtypes = [ctypes.c_void_p]
        lib.orc_set_solid.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.orc_set_fields.argtypes = [ctypes.c_void_p, dp, dp, dp]
        lib.orc_set_populations.argtypes = [ctypes.c_void_p, dp, dp, dp]
        lib.orc_get_populations.argtypes = [ctypes.c_void_p, dp, dp, dp]
        lib.orc_step.argtypes = [ctypes.c_void_p, ctypes.c_long]
        lib.orc_step_push_ghost.argtypes = [ctypes.c_void_p, ctypes.c_long]
        lib.orc_fields.argtypes = [ctypes.c_void_p, dp, dp, dp, dp]
        lib.orc_forces.argtypes = [ctypes.c_void_p, dp, dp]
        lib.orc_observables.argtypes = [ctypes.c_void_p, dp]
        lib.orc_x_average.argtypes = [ctypes.c_void_p, dp]
        lib.orc_stress_xy.argtypes = [ctypes.c_void_p, dp]
        lib.orc_row_average.argtypes = [ctypes.c_void_p, dp, dp]
        lib.orc_row_momentum_x.argtypes = [ctypes.c_void_p, dp]
        lib.orc_droplets.restype = ctypes.c_int
        lib.orc_droplets.argtypes = [ctypes.c_void_p, ctypes.c_double, ctypes.c_void_p, ctypes.c_int, dp]
        i32p = ctypes.c_void_p
        lib.orc_voronoi.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, ctypes.c_int, i32p]
        lib.orc_voronoi_at.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, ctypes.c_int, i32p, ctypes.c_int, i32p]
        lib.orc_delaunay.restype = ctypes.c_int
        lib.orc_delaunay.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, i32p, ctypes.c_int, i32p]
        lib.orc_match.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, i32p, dp, ctypes.c_int, i32p]
        lib.orc_displacements.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, i32p, ctypes.c_int, dp]
        lib.orc_t1_events.restype = ctypes.c_int
        lib.orc_t1_events.argtypes = [i32p, ctypes.c_int, i32p, ctypes.c_int, i32p, ctypes.c_int, i32p]
        lib.orc_droplet_nusselt.argtypes = [ctypes.c_void_p, dp, ctypes.c_int, dp]
        lib.orc_rough_walls.argtypes = [ctypes.c_int] * 7 + [ctypes.c_double, ctypes.c_int, ctypes.c_void_p]
        lib.orc_perturb_velocity.argtypes = [ctypes.c_void_p, ctypes.c_double]
        lib.orc_w.restype = ctypes.c_double
        lib.orc_w.argtypes = [ctypes.c_int, ctypes.c_int]
        lib.orc_p.restype = ctypes.c_double
        lib.orc_p.argtypes = [ctypes.c_int, ctypes.c_int]
        lib.orc_direction.argtypes = [ctypes.c_int] + [ctypes.POINTER(ctypes.c_int)] * 3
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _c(a):
    return np.ascontiguousarray(a, dtype=np.float64)


# parameter names understood by Oracle(**params); anything else (init recipe, posts) is ignored
PARAM_KEYS = [n for n, _ in OrcParams._fields_]


class Oracle:
    """One lattice of nx x ny sites.  Arrays are [ny][nx] (x fastest); populations [9][ny][nx]."""

    def __init__(self, nx, ny, **params):
        self.lib = _load()
        self.nx, self.ny = int(nx), int(ny)
        p = OrcParams()
        defaults = dict(tau=1.0, tau_g=1.0, rho0=1.0, G12=0.0, G11a=0.0, G11r=0.0, G22a=0.0, G22r=0.0,
                        rho_wall_A=0.0, rho_wall_B=0.0, T_bottom=0.0, T_top=0.0, T_ref=0.0, alpha_g=0.0,
                        body_ax=0.0, u_wall_bottom=0.0, u_wall_top=0.0, periodic_y=0, thermal=1)
        for k in PARAM_KEYS:
            setattr(p, k, params.get(k, defaults[k]))
        self.params = p
        self.h = self.lib.orc_create(self.nx, self.ny, ctypes.byref(p))
        if not self.h:
            raise ValueError("orc_create failed")

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.orc_destroy(self.h)
            self.h = None

    def set_solid(self, solid):
        s = np.ascontiguousarray(solid, dtype=np.uint8)
        assert s.shape == (self.ny, self.nx)
        self.lib.orc_set_solid(self.h, s.ctypes.data)

    def set_fields(self, rhoA, rhoB, T):
        a, b, t = _c(rhoA), _c(rhoB), _c(T)
        assert a.shape == b.shape == t.shape == (self.ny, self.nx)
        self.lib.orc_set_fields(self.h, _dp(a), _dp(b), _dp(t))

    def set_populations(self, fA, fB, g):
        a, b, c = _c(fA), _c(fB), _c(g)
        assert a.shape == (9, self.ny, self.nx)
        self.lib.orc_set_populations(self.h, _dp(a), _dp(b), _dp(c))

    def get_populations(self):
        out = [np.empty((9, self.ny, self.nx)) for _ in range(3)]
        self.lib.orc_get_populations(self.h, *[_dp(o) for o in out])
        return out

    def step(self, n=1):
        self.lib.orc_step(self.h, int(n))

    def step_push_ghost(self, n=1):
        self.lib.orc_step_push_ghost(self.h, int(n))

    def fields(self):
        rhoA, rhoB, T = (np.empty((self.ny, self.nx)) for _ in range(3))
        u = np.empty((2, self.ny, self.nx))
        self.lib.orc_fields(self.h, _dp(rhoA), _dp(rhoB), _dp(u), _dp(T))
        return rhoA, rhoB, u, T

    def forces(self):
        FA, FB = np.empty((2, self.ny, self.nx)), np.empty((2, self.ny, self.nx))
        self.lib.orc_forces(self.h, _dp(FA), _dp(FB))
        return FA, FB

    def observables(self):
        out = np.empty(4)
        self.lib.orc_observables(self.h, _dp(out))
        return dict(mass_A=out[0], mass_B=out[1], E=out[2], Nu=out[3])


def _x_average(self):
    """u_av[y]: x-average of u_x^(H) over the fluid sites of each row."""
    out = np.empty(self.ny)
    self.lib.orc_x_average(self.h, _dp(out))
    return out


Oracle.x_average = _x_average


def _stress_xy(self):
    """P_xy [ny][nx] (reading R21)."""
    out = np.empty((self.ny, self.nx))
    self.lib.orc_stress_xy(self.h, _dp(out))
    return out


def _x_average_stress(self):
    """Pxy_av[ny]: x-average of P_xy over the fluid sites of each row."""
    pxy = _stress_xy(self)
    out = np.empty(self.ny)
    self.lib.orc_row_average(self.h, _dp(pxy), _dp(out))
    return out


def _row_momentum_x(self):
    out = np.empty(self.ny)
    self.lib.orc_row_momentum_x(self.h, _dp(out))
    return out


def _droplets(self, B_th, max_droplets):
    """(labels [ny][nx] int32, n_droplets, stats [min(n, max)][4]) -- section 2.4, reading R22."""
    labels = np.empty((self.ny, self.nx), dtype=np.int32)
    stats = np.zeros((max(1, max_droplets), 4))
    n = self.lib.orc_droplets(self.h, float(B_th), labels.ctypes.data, int(max_droplets), _dp(stats))
    return labels, n, stats[:min(n, max_droplets)]


Oracle.stress_xy = _stress_xy
Oracle.x_average_stress = _x_average_stress
Oracle.row_momentum_x = _row_momentum_x
Oracle.droplets = _droplets


def _droplet_nusselt(self, centres):
    """Nu_i of Eq. (25) at the lattice site nearest to each centre [n][2] (reading R26)."""
    c = _c(centres).reshape(-1, 2)
    nu = np.zeros(len(c))
    self.lib.orc_droplet_nusselt(self.h, _dp(c), len(c), _dp(nu))
    return nu


Oracle.droplet_nusselt = _droplet_nusselt


def _perturb_velocity(self, amplitude):
    """One roll pair of amplitude A added to both fluids' momentum (reading R29)."""
    self.lib.orc_perturb_velocity(self.h, float(amplitude))


Oracle.perturb_velocity = _perturb_velocity


def rough_walls(nx, ny, up, down, width, height, lam, alpha, asymmetric):
    """Obstacle mask [ny][nx] uint8 of trapezoidal rough walls (reading R27)."""
    solid = np.zeros((ny, nx), dtype=np.uint8)
    _load().orc_rough_walls(int(nx), int(ny), int(up), int(down), int(width), int(height), int(lam), float(alpha),
                            int(asymmetric), solid.ctypes.data)
    return solid


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def voronoi(nx, ny, periodic_y, centres):
    """Digital Voronoi colouring [ny][nx] int32 of the centres [n][2] (reading R23); brute force."""
    c = _c(centres).reshape(-1, 2)
    colour = np.zeros((ny, nx), dtype=np.int32)
    _load().orc_voronoi(int(nx), int(ny), int(bool(periodic_y)), _dp(c), len(c), colour.ctypes.data)
    return colour


def voronoi_at(nx, ny, periodic_y, centres, sites):
    """Colours of the listed sites (y nx + x) only; the same brute force as voronoi()."""
    c = _c(centres).reshape(-1, 2)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.zeros(len(sites), dtype=np.int32)
    _load().orc_voronoi_at(int(nx), int(ny), int(bool(periodic_y)), _dp(c), len(c), sites.ctypes.data, len(sites), out.ctypes.data)
    return out


def delaunay(colour, periodic_y, max_links=None):
    """Sorted distinct Delaunay links [m][2] of a colouring (reading R24)."""
    colour = _i32(colour)
    ny, nx = colour.shape
    cap = int(max_links) if max_links is not None else 16 * (int(colour.max()) + 2)
    links = np.zeros((max(cap, 1), 2), dtype=np.int32)
    n = _load().orc_delaunay(nx, ny, int(bool(periodic_y)), colour.ctypes.data, cap, links.ctypes.data)
    return links[:min(n, cap)].copy(), n


def match(colour_past, periodic_y, centres_now):
    """map[i] = past droplet in whose Voronoi cell the present centre i lies (reading R25)."""
    colour_past = _i32(colour_past)
    ny, nx = colour_past.shape
    c = _c(centres_now).reshape(-1, 2)
    m = np.zeros(len(c), dtype=np.int32)
    _load().orc_match(nx, ny, int(bool(periodic_y)), colour_past.ctypes.data, _dp(c), len(c), m.ctypes.data)
    return m


def displacements(nx, ny, periodic_y, centres_past, centres_now, map_now_to_past):
    """d_i = X_i(now) - X_map[i](past) in minimum image, [n_now][2]; (0, 0) for unmatched droplets."""
    cp, cn = _c(centres_past).reshape(-1, 2), _c(centres_now).reshape(-1, 2)
    mp = _i32(map_now_to_past)
    out = np.zeros((len(cn), 2))
    _load().orc_displacements(int(nx), int(ny), int(bool(periodic_y)), _dp(cp), _dp(cn), mp.ctypes.data, len(cn), _dp(out))
    return out


def t1_events(links_past, links_now, map_now_to_past=None, max_events=4096):
    """T1 events [e][4] = (a, b, c, d): link a-b replaced by link c-d (reading R25)."""
    lp, ln = _i32(links_past).reshape(-1, 2), _i32(links_now).reshape(-1, 2)
    mp = _i32(map_now_to_past) if map_now_to_past is not None else None
    ev = np.zeros((max(max_events, 1), 4), dtype=np.int32)
    n = _load().orc_t1_events(lp.ctypes.data, len(lp), ln.ctypes.data, len(ln), mp.ctypes.data if mp is not None else None,
                              int(max_events), ev.ctypes.data)
    return ev[:min(n, max_events)].copy(), n


def lattice_weights():
    """(w, p) of Fig. 1(b) as dicts {(dx, dy): weight} over the 5x5 neighbourhood."""
    lib = _load()
    w = {(dx, dy): lib.orc_w(dx, dy) for dx in range(-2, 3) for dy in range(-2, 3)}
    p = {(dx, dy): lib.orc_p(dx, dy) for dx in range(-2, 3) for dy in range(-2, 3)}
    return w, p


def directions():
    lib = _load()
    out = []
    for i in range(9):
        cx, cy, op = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
        lib.orc_direction(i, ctypes.byref(cx), ctypes.byref(cy), ctypes.byref(op))
        out.append((cx.value, cy.value, op.value))
    return out
