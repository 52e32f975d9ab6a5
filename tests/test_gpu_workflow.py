"""GPU parity of the workflow pieces: trapezoidal rough walls (R27, PAPER section 4), the honeycomb
droplet initialisation (L266), the initial velocity perturbation (R29, L322) and the binary population dumps / restart
(Table C.11).  Through the C ABI, against the oracle and the shared input generators."""
import os

import numpy as np
import pytest

import inputs
pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def tlbmod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2109_12565_b200 import binding
    binding.load_library()
    return binding


def _np(t):
    return t.cpu().numpy()


@pytest.mark.parametrize("nx,ny,up,down,w,h,lam,alpha,asym", [
    (300, 60, 1, 1, 10, 9, 150, 0.25, 1),      # Table A.6
    (300, 60, 1, 1, 10, 9, 150, 0.25, 0),
    (250, 37, 0, 1, 12, 6, 25, 0.6, 0),        # several strips + ragged tail, bottom wall only, steep sides
    (128, 32, 1, 0, 6, 5, 16, np.pi / 4, 1),   # tan(alpha) rounds next to 1: floor(j tan) is taken on the host on both sides
    (64, 24, 1, 1, 4, 4, 16, 0.0, 0),          # rectangles = the posts of config 4
])
def test_rough_walls_mask_and_run(tlbmod, oracle_mod, nx, ny, up, down, w, h, lam, alpha, asym):
    """The mask is read back through tlb_fields (solid sites report rho_wall_A, here a sentinel) and must equal the
    oracle's; then 10 steps on that geometry against the oracle."""
    par = dict(inputs.PAPER_PHYSICS, alpha_g=1e-4, rho_wall_A=7.25, rho_wall_B=0.3)
    solid = oracle_mod.rough_walls(nx, ny, up, down, w, h, lam, alpha, asym)
    t = tlbmod.TLB(nx, ny, **par)
    t.set_rough_walls(up, down, w, h, lam, alpha, asym)
    rA, rB, T = inputs.smooth_random_fields(nx, ny, 4, 0.5, -0.5)
    t.set_fields(rA, rB, T)
    assert ((_np(t.fields()[0]) == 7.25) == (solid == 1)).all()
    o = oracle_mod.Oracle(nx, ny, **par)
    o.set_solid(solid)
    o.set_fields(rA, rB, T)
    t.step(10)
    o.step(10)
    assert max(np.abs(a - _np(b)).max() for a, b in zip(o.get_populations(), t.get_populations())) <= TOL
    if alpha == 0.0:
        assert (solid == inputs.post_mask(nx, ny, w, h, lam)).all()


def test_rough_walls_errors(tlbmod):
    t = tlbmod.TLB(64, 16)
    for args in ((1, 1, 4, 9, 16, 0.1, 0), (1, 1, 20, 3, 16, 0.1, 0), (1, 1, 4, 3, 0, 0.1, 0)):
        with pytest.raises(tlbmod.TLBError):
            t.set_rough_walls(*args)
    tp = tlbmod.TLB(64, 16, periodic_y=1)
    with pytest.raises(tlbmod.TLBError):
        tp.set_rough_walls(1, 1, 4, 3, 16, 0.1, 0)


@pytest.mark.parametrize("nx,ny,ndx,ndy,posts", [(128, 64, 6, 4, (0, 0, 0)), (250, 96, 7, 5, (4, 4, 16)), (512, 256, 20, 10, (0, 0, 0))])
def test_init_honeycomb_bit_identical(tlbmod, nx, ny, ndx, ndy, posts):
    """tlb_init_honeycomb against inputs.honeycomb_centres + inputs.initial_fields passed through tlb_set_fields: the
    populations must be bit-identical (as for tlb_init)."""
    cfg = dict(inputs.config(1, "paper"), nx=nx, ny=ny, posts=posts)
    ini, p = cfg["init"], cfg["params"]
    r = min(ini["droplet_radius"], 0.3 * min(nx / ndx, (ny - 2 * posts[1]) / ndy))
    cfg["init"] = dict(ini, droplet_radius=r)
    solid = inputs.post_mask(nx, ny, *posts)
    cen = inputs.honeycomb_centres(nx, ny, ndx, ndy, post_h=posts[1])
    rA, rB, T = inputs.initial_fields(nx, ny, 9, 0, r, 0.0, ini["rho_in"], ini["rho_out"], ini["noise_amp"],
                                      p["T_bottom"], p["T_top"], solid=solid, post_h=posts[1], centres=cen)
    assert (rA > 0.5 * (ini["rho_in"] + ini["rho_out"])).sum() > 0.5 * ndx * ndy * np.pi * r * r
    t = tlbmod.TLB(nx, ny, params=tlbmod.params_from_config(cfg))
    t.init_honeycomb(ndx, ndy, 9)
    t2 = tlbmod.TLB(nx, ny, params=tlbmod.params_from_config(cfg))
    t2.set_solid(solid)
    t2.set_fields(rA, rB, T)
    for a, b in zip(t.get_populations(), t2.get_populations()):
        assert bool((a == b).all())
    # the droplet analysis finds the ndx * ndy discs where the generator put them
    B_th = 0.5 * (ini["rho_in"] + ini["rho_out"])
    _, k, stats = t.droplets(B_th, 4 * ndx * ndy)
    assert k == ndx * ndy
    got = _np(stats)[:, 2:4]
    d = got[:, None, :] - cen[None, :, :]
    d[..., 0] -= nx * np.round(d[..., 0] / nx)
    assert np.sqrt((d ** 2).sum(-1)).min(1).max() < 0.75


@pytest.mark.parametrize("geom", ["walls", "posts"])
def test_perturb_velocity_parity(tlbmod, oracle_mod, geom):
    nx, ny, A = 200, 46, 1e-3
    par = dict(inputs.PAPER_PHYSICS, alpha_g=1e-4)
    solid = inputs.post_mask(nx, ny, 4, 4, 16) if geom == "posts" else np.zeros((ny, nx), np.uint8)
    rA, rB, T = inputs.smooth_random_fields(nx, ny, 6, 0.5, -0.5)
    t = tlbmod.TLB(nx, ny, **par)
    o = oracle_mod.Oracle(nx, ny, **par)
    for s in (t, o):
        s.set_solid(solid)
        s.set_fields(rA, rB, T)
    t.step(3)
    o.step(3)
    m0 = t.observables()
    t.perturb_velocity(A)
    o.perturb_velocity(A)
    d = max(np.abs(a - _np(b)).max() for a, b in zip(o.get_populations(), t.get_populations()))
    assert d <= 1e-15
    m1 = t.observables()
    assert abs(m1["mass_A"] / m0["mass_A"] - 1) < 1e-14 and abs(m1["mass_B"] / m0["mass_B"] - 1) < 1e-14
    assert m1["E"] != m0["E"] and m1["E"] == pytest.approx(o.observables()["E"], rel=1e-12)
    t.step(10)
    o.step(10)
    assert max(np.abs(a - _np(b)).max() for a, b in zip(o.get_populations(), t.get_populations())) <= TOL
    with pytest.raises(tlbmod.TLBError):
        tlbmod.TLB(32, 16).perturb_velocity(A)   # no state yet


@pytest.mark.parametrize("prec", [64, 32])
def test_checkpoint_restart(tlbmod, oracle_mod, tmp_path, prec):
    """Dump after 7 steps, restore into a fresh handle, run both 9 more steps: bit-identical.  The files are the raw
    [9][ny][nx] fp64 arrays of tlb_get_populations; the oracle restarted from the same files stays within 1e-12."""
    cfg = dict(inputs.config(1, "paper"), posts=(4, 4, 16))
    nx, ny = cfg["nx"], cfg["ny"]
    par = tlbmod.params_from_config(cfg)
    par.pop_precision = prec
    solid, rA, rB, T = inputs.make_config_inputs(cfg)
    t = tlbmod.TLB(nx, ny, params=par)
    t.init(cfg["seed"])
    t.step(7)
    d = str(tmp_path)
    t.write_checkpoint(d, 3)
    pops = [_np(p) for p in t.get_populations()]
    for stem, p in zip(("conf1", "conf2", "confG"), pops):
        f = os.path.join(d, "%s_3.in" % stem)
        assert os.path.getsize(f) == 9 * nx * ny * 8
        assert (np.fromfile(f, dtype="<f8").reshape(9, ny, nx) == p).all()
    t2 = tlbmod.TLB(nx, ny, params=par)
    t2.set_solid(solid)
    t2.read_checkpoint(d, 3)
    t.step(9)
    t2.step(9)
    for a, b in zip(t.get_populations(), t2.get_populations()):
        assert bool((a == b).all())
    if prec == 64:
        o = oracle_mod.Oracle(nx, ny, **cfg["params"])
        o.set_solid(solid)
        o.set_populations(*[np.fromfile(os.path.join(d, "%s_3.in" % s), dtype="<f8").reshape(9, ny, nx) for s in ("conf1", "conf2", "confG")])
        o.step(9)
        assert max(np.abs(a - _np(b)).max() for a, b in zip(o.get_populations(), t2.get_populations())) <= TOL
    # errors: a missing index, a dump of another lattice size
    with pytest.raises(tlbmod.TLBError) as e:
        t2.read_checkpoint(d, 4)
    assert e.value.code == tlbmod.TLB_EIO
    t3 = tlbmod.TLB(nx // 2, ny, params=par)
    with pytest.raises(tlbmod.TLBError) as e:
        t3.read_checkpoint(d, 3)
    assert e.value.code == tlbmod.TLB_EIO


def test_write_fields_round_trip(tlbmod, tmp_path):
    """Tables C.9 / C.10 (reading R31): the ASCII files read back to exactly the arrays of tlb_fields, tlb_x_average,
    tlb_stress_xy and tlb_x_average_stress (17 significant digits), in the documented order; the .vtk twins are
    binary legacy VTK 2.0 STRUCTURED_POINTS whose big-endian doubles are those arrays."""
    cfg = dict(inputs.config(1, "paper"), nx=96, ny=40, posts=(4, 4, 16))
    cfg["init"] = dict(cfg["init"], n_droplets=5)
    nx, ny = cfg["nx"], cfg["ny"]
    t = tlbmod.TLB(nx, ny, params=tlbmod.params_from_config(cfg))
    t.init(3)
    t.step(25)
    d = str(tmp_path)
    t.write_fields(d, 7, what=15, vtk=True)
    rA, rB, u, T = [_np(a) for a in t.fields()]
    expect = {"firstdensity": [rA], "seconddensity": [rB], "temperature": [T], "veloconf": [u[0], u[1]], "Ptot_xy": [_np(t.stress_xy())]}
    X, Y = np.meshgrid(np.arange(nx), np.arange(ny))
    for name, arrs in expect.items():
        m = np.loadtxt(os.path.join(d, "%s.7.dat" % name))
        assert m.shape == (nx * ny, 2 + len(arrs))
        assert (m[:, 0] == X.ravel()).all() and (m[:, 1] == Y.ravel()).all()
        for k, a in enumerate(arrs):
            assert (m[:, 2 + k] == a.ravel()).all(), name
        raw = open(os.path.join(d, "%s.7.dat" % name)).read().split("\n")
        assert raw[nx] == "" and raw[nx + 1].startswith("0 1 ")          # a blank line after every lattice row
        blob = open(os.path.join(d, "%s.7.vtk" % name), "rb").read()
        n_head = 9 if len(arrs) == 2 else 10
        head = blob.split(b"\n", n_head)[:n_head]
        assert head[0] == b"# vtk DataFile Version 2.0" and head[2] == b"BINARY"                    # L244-246
        assert head[3] == b"DATASET STRUCTURED_POINTS" and head[4] == b"DIMENSIONS %d %d 1" % (nx, ny)
        assert head[8] == (b"VECTORS %s double" if len(arrs) == 2 else b"SCALARS %s double 1") % name.encode()
        body = blob[sum(len(h) + 1 for h in head):]
        vals = np.frombuffer(body[:-1], dtype=">f8").reshape(nx * ny, -1)                             # big-endian doubles
        assert body[-1:] == b"\n" and vals.shape[1] == (3 if len(arrs) == 2 else 1)
        for k, a in enumerate(arrs):
            assert (vals[:, k] == a.ravel()).all(), name
    for name, a in (("u_av", _np(t.x_average())), ("Pxy_av", _np(t.x_average_stress()))):
        m = np.loadtxt(os.path.join(d, "%s.7.dat" % name))
        assert m.shape == (ny, 2) and (m[:, 0] == np.arange(ny)).all() and (m[:, 1] == a).all()
    # only what was asked for is written
    t.write_fields(d, 8, what=t.OUT_TEMPERATURE)
    assert sorted(f for f in os.listdir(d) if ".8." in f) == ["temperature.8.dat"]
    # timeEnergy.dat (L248): one "<index> E" line appended per call, E the observable, 17 digits
    assert not os.path.exists(os.path.join(d, "timeEnergy.dat"))
    e25 = t.observables()["E"]
    t.write_fields(d, 25, what=t.OUT_ENERGY)
    t.step(5)
    t.write_fields(d, 30, what=t.OUT_ENERGY)
    rows = np.loadtxt(os.path.join(d, "timeEnergy.dat"))
    assert rows.shape == (2, 2) and (rows[:, 0] == [25, 30]).all()
    assert rows[0, 1] == e25 and rows[1, 1] == t.observables()["E"] and e25 > 0
    with pytest.raises(tlbmod.TLBError) as e:
        t.write_fields(os.path.join(d, "missing"), 9)
    assert e.value.code == tlbmod.TLB_EIO


def test_bench_json_contract(tlbmod):
    """bench.py prints ONE JSON line with the keys the driver reads (small config, short run)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--config", "1", "--steps", "20", "--warmup", "3"],
                         capture_output=True, text=True, timeout=600, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert key in d, key
    assert d["metric"] == "MLUPS" and d["unit"] == "MLUPS" and d["n_gpus"] == 1 and d["steps"] == 20 and d["dtype"] == "f64"
    assert d["higher_is_better"] is True and d["vs_baseline"] is None and d["data"] == "synthetic"
    assert d["config"]["workload"].startswith("config1") and "model" not in d["config"]
    assert d["gpu_launches"] == 40 and d["value"] > 0
    r = d["roofline"]
    for key in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert key in r, key
    assert r["bound"] == "hbm" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] == 1 and c["value"] > 0 and "sample" in c
    e = d["e2e"]   # the loop that returns the step's result: three field planes in, five out
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 3 * 8 * 128 * 64 and e["d2h_bytes_per_step"] == 5 * 8 * 128 * 64
    assert d["e2e_observables"]["d2h_bytes_per_step"] == 32 and d["e2e_observables"]["value"] > e["value"]
    sus = r["sustained"]   # the config's own step count (config 1: 1000), timed after the K-step region
    assert sus["steps"] == 1000 and sus["ms_per_step"] > 0 and sus["frac"] > 0 and "clocks" in sus
    assert d["droplet_analysis"]["n_droplets"] == 12 and d["droplet_analysis"]["whole_analysis_lb_steps"] > 0
    assert d["scaling"] == "strong"
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
