"""Thin ctypes binding of the C ABI in include/tlb.h (same names, argument marshalling only).

Every step of the path runs in the CUDA kernels of csrc/; PyTorch is used for device memory and
streams.  There is no CPU fallback: if libtlb.so is missing or no CUDA device is present the calls
raise.  This module never imports anything under oracle/.
"""
import ctypes
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB_PATH = os.path.join(_HERE, "libtlb.so")
SOURCES = ["tlb_step.cu", "tlb_aux.cu", "tlb_analysis.cu", "tlb_api.cu", "tlb_noalloc.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC,-ffp-contract=off", "-shared"]

TLB_OK, TLB_EINVAL, TLB_ESTATE, TLB_ECUDA, TLB_EPLACEMENT, TLB_EIO, TLB_ELIMIT = 0, -1, -2, -3, -4, -5, -6
T1_STATIC_MAX_DROPLETS = T1_STATIC_MAX_EVENTS = 16384  # TLB_T1_STATIC_MAX_* of include/tlb.h

# every symbol include/tlb.h declares
SYMBOLS = ["tlb_default_params", "tlb_workspace_bytes", "tlb_create", "tlb_destroy", "tlb_slab_workspace_bytes",
           "tlb_create_slab", "tlb_slab_layout", "tlb_halo_bytes", "tlb_seg_rows", "tlb_init", "tlb_init_honeycomb",
           "tlb_set_rough_walls", "tlb_perturb_velocity", "tlb_write_checkpoint", "tlb_read_checkpoint", "tlb_write_fields", "tlb_set_solid",
           "tlb_set_solid_host", "tlb_set_fields", "tlb_set_fields_host", "tlb_set_populations",
           "tlb_get_populations", "tlb_set_populations_host", "tlb_get_populations_host", "tlb_step",
           "tlb_slab_step_edges", "tlb_slab_step_interior", "tlb_slab_step_finish", "tlb_halo_pack", "tlb_halo_unpack",
           "tlb_halo_region",
           "tlb_profile_step", "tlb_fields", "tlb_fields_host", "tlb_observables", "tlb_observables_host",
           "tlb_observable_sums", "tlb_observables_from_sums", "tlb_x_average", "tlb_x_average_host",
           "tlb_stress_xy", "tlb_stress_xy_host", "tlb_x_average_stress", "tlb_x_average_stress_host",
           "tlb_droplets", "tlb_droplets_host", "tlb_voronoi", "tlb_delaunay", "tlb_droplet_match", "tlb_droplet_displacements", "tlb_t1_events",
           "tlb_t1_events_static",
           "tlb_droplet_nusselt", "tlb_launch_count", "tlb_error_string", "tlb_last_cuda_error"]


class TLBParams(ctypes.Structure):
    """Mirror of `struct tlb_params` (include/tlb.h)."""
    _fields_ = [(n, ctypes.c_double) for n in (
        "tau", "tau_g", "rho0", "G12", "G11a", "G11r", "G22a", "G22r", "rho_wall_A", "rho_wall_B",
        "T_bottom", "T_top", "T_ref", "alpha_g", "body_ax", "u_wall_bottom", "u_wall_top",
        "droplet_radius", "min_gap", "rho_in", "rho_out", "noise_amp")] + [(n, ctypes.c_int32) for n in (
            "n_droplets", "periodic_y", "thermal", "post_w", "post_h", "post_period", "pop_precision", "reserved")]


class TLBRoughWalls(ctypes.Structure):
    """Mirror of `struct tlb_rough_walls` (include/tlb.h)."""
    _fields_ = [("alpha", ctypes.c_double)] + [(n, ctypes.c_int32) for n in ("up", "down", "width", "height", "lam", "asymmetric")]


class TLBError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("tlb error %d: %s" % (code, msg))
        self.code = code


def _sources_newer():
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    deps = [os.path.join(_CSRC, s) for s in SOURCES] + [os.path.join(_CSRC, "tlb_internal.cuh"),
                                                        os.path.join(_INCLUDE, "tlb.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    """Compile csrc/*.cu for sm_100a into paper_2109_12565_b200/libtlb.so (in-tree)."""
    if not force and not _sources_newer():
        return LIB_PATH
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB_PATH + ".%d.tmp" % os.getpid()
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-I", _INCLUDE, "-o", tmp] + \
          [os.path.join(_CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB_PATH)
    return LIB_PATH


_lib = None


def load_library():
    """dlopen libtlb.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise TLBError(TLB_ECUDA, "libtlb.so is not built (run __graft_entry__.build()); there is no CPU fallback")
    lib = ctypes.CDLL(LIB_PATH)
    vp, dp, i32, i64 = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int64
    pp = ctypes.POINTER(TLBParams)
    lib.tlb_default_params.argtypes = [pp]
    lib.tlb_workspace_bytes.argtypes = [i32, i32, pp, ctypes.POINTER(ctypes.c_size_t)]
    lib.tlb_create.argtypes = [i32, i32, pp, vp, ctypes.c_size_t, vp, ctypes.POINTER(vp)]
    lib.tlb_destroy.argtypes = [vp]
    lib.tlb_init.argtypes = [vp, ctypes.c_uint64]
    lib.tlb_init_honeycomb.argtypes = [vp, i32, i32, ctypes.c_uint64]
    lib.tlb_set_rough_walls.argtypes = [vp, ctypes.POINTER(TLBRoughWalls)]
    lib.tlb_perturb_velocity.argtypes = [vp, ctypes.c_double]
    lib.tlb_write_checkpoint.argtypes = [vp, ctypes.c_char_p, i32]
    lib.tlb_read_checkpoint.argtypes = [vp, ctypes.c_char_p, i32]
    lib.tlb_write_fields.argtypes = [vp, ctypes.c_char_p, i32, i32, i32]
    lib.tlb_set_solid.argtypes = [vp, dp]
    lib.tlb_set_solid_host.argtypes = [vp, dp]
    for name in ("tlb_set_fields", "tlb_set_fields_host", "tlb_set_populations", "tlb_get_populations",
                 "tlb_set_populations_host", "tlb_get_populations_host"):
        getattr(lib, name).argtypes = [vp, dp, dp, dp]
    lib.tlb_step.argtypes = [vp, i64]
    lib.tlb_profile_step.argtypes = [vp, i64, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    lib.tlb_fields.argtypes = [vp, dp, dp, dp, dp]
    lib.tlb_fields_host.argtypes = [vp, dp, dp, dp, dp]
    lib.tlb_observables.argtypes = [vp, dp]
    lib.tlb_observables_host.argtypes = [vp, dp]
    for name in ("tlb_x_average", "tlb_x_average_host", "tlb_stress_xy", "tlb_stress_xy_host", "tlb_x_average_stress",
                 "tlb_x_average_stress_host", "tlb_observable_sums"):
        getattr(lib, name).argtypes = [vp, dp]
    lib.tlb_observables_from_sums.argtypes = [vp, dp, dp]
    lib.tlb_slab_workspace_bytes.argtypes = [i32, i32, i32, i32, pp, ctypes.POINTER(ctypes.c_size_t)]
    lib.tlb_create_slab.argtypes = [i32, i32, i32, i32, pp, vp, ctypes.c_size_t, vp, ctypes.POINTER(vp)]
    lib.tlb_slab_layout.argtypes = [vp, ctypes.POINTER(ctypes.c_int32)]
    lib.tlb_halo_bytes.argtypes = [vp, ctypes.POINTER(ctypes.c_size_t)]
    lib.tlb_seg_rows.argtypes = [vp]
    for name in ("tlb_slab_step_edges", "tlb_slab_step_interior", "tlb_slab_step_finish"):
        getattr(lib, name).argtypes = [vp]
    lib.tlb_halo_region.argtypes = [vp, i32, i32, ctypes.POINTER(ctypes.c_void_p), ctypes.POINTER(ctypes.c_size_t)]
    lib.tlb_halo_pack.argtypes = [vp, i32, dp]
    lib.tlb_halo_unpack.argtypes = [vp, i32, dp]
    lib.tlb_droplets.argtypes = [vp, ctypes.c_double, dp, i32, dp, dp]
    lib.tlb_droplets_host.argtypes = [vp, ctypes.c_double, dp, i32, dp, dp]
    lib.tlb_voronoi.argtypes = [vp, dp, i32, dp]
    lib.tlb_delaunay.argtypes = [vp, dp, i32, i32, dp, dp]
    lib.tlb_droplet_match.argtypes = [vp, dp, dp, i32, dp]
    lib.tlb_droplet_displacements.argtypes = [vp, dp, dp, dp, i32, dp]
    lib.tlb_t1_events.argtypes = [vp, dp, i32, dp, i32, dp, i32, i32, i32, dp, dp]
    lib.tlb_t1_events_static.argtypes = [dp, i32, dp, i32, dp, i32, i32, i32, dp, dp, vp]
    lib.tlb_droplet_nusselt.argtypes = [vp, dp, i32, dp]
    lib.tlb_launch_count.argtypes = [vp]
    lib.tlb_launch_count.restype = i64
    lib.tlb_error_string.argtypes = [i32]
    lib.tlb_error_string.restype = ctypes.c_char_p
    lib.tlb_last_cuda_error.argtypes = [vp]
    lib.tlb_last_cuda_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


def default_params(**overrides):
    """tlb_default_params() with keyword overrides; unknown keys raise."""
    p = TLBParams()
    load_library().tlb_default_params(ctypes.byref(p))
    names = {n for n, _ in TLBParams._fields_}
    for k, v in overrides.items():
        if k not in names:
            raise KeyError(k)
        setattr(p, k, v)
    return p


def _ptr(t):
    return None if t is None else t.data_ptr()


def t1_events_static(links_past, links_now, n_droplets, n_events, events, map_now_to_past=None, stream=None):
    """tlb_t1_events_static: the T1 events between two Delaunay link lists without a TLB handle, a workspace or any
    device allocation -- for tools that own no lattice, for monitors running beside a lattice that fills the GPU, and for
    hosts that do not let guests allocate (include/tlb.h has the full story).  Nothing is allocated here either: the
    caller passes the outputs, `n_events` (int32 [1]) and `events` (int32 [max_events][4]), next to the inputs
    (contiguous int32 CUDA tensors on one device; `map_now_to_past` may be None).  The work goes on `stream` (default:
    torch's current stream of that device) and is not synchronised.  At most T1_STATIC_MAX_DROPLETS droplets
    (TLBError with code TLB_ELIMIT beyond).  All calls on one GPU share one scratch array: do not let two overlap."""
    import torch
    lib = load_library()
    tensors = [t for t in (links_past, links_now, map_now_to_past, n_events, events) if t is not None]
    for t in tensors:
        if t.dtype != torch.int32 or not t.is_cuda or not t.is_contiguous() or t.device != n_events.device:
            raise TLBError(TLB_EINVAL, "t1_events_static takes contiguous int32 CUDA tensors on one device")
    if n_events.numel() < 1 or (events.numel() > 0 and (events.dim() != 2 or events.shape[1] != 4)):
        raise TLBError(TLB_EINVAL, "n_events is int32 [1], events is int32 [max_events][4]")
    with torch.cuda.device(n_events.device):  # the entry point works on the current device
        st = stream if stream is not None else torch.cuda.current_stream()
        rc = lib.tlb_t1_events_static(_ptr(links_past), int(links_past.shape[0]), _ptr(links_now), int(links_now.shape[0]),
                                      _ptr(map_now_to_past), 0 if map_now_to_past is None else int(map_now_to_past.shape[0]),
                                      int(n_droplets), int(events.shape[0]), n_events.data_ptr(), _ptr(events), st.cuda_stream)
    if rc != TLB_OK:
        raise TLBError(rc, lib.tlb_error_string(rc).decode())


class TLB:
    """One lattice on one GPU.  Methods mirror the C calls; tensors are torch CUDA float64 (device
    variants) or CPU float64 (the *_host variants; pin them for asynchronous copies)."""

    def __init__(self, nx, ny, params=None, device="cuda:0", stream=None, slab=None, **overrides):
        """slab = (y0, y1): a y-slab handle for rows [y0, y1) of the nx x ny lattice (tlb_create_slab); self.ny is
        then the number of local rows (owned + halo) and self.ny_global the lattice's."""
        import torch
        self.torch = torch
        self.lib = load_library()
        self.nx, self.ny_global = int(nx), int(ny)
        self.params = params if params is not None else default_params(**overrides)
        if params is not None:
            for k, v in overrides.items():
                setattr(self.params, k, v)
        nbytes = ctypes.c_size_t()
        if slab is None:
            self._chk(self.lib.tlb_workspace_bytes(self.nx, self.ny_global, ctypes.byref(self.params), ctypes.byref(nbytes)))
        else:
            self._chk(self.lib.tlb_slab_workspace_bytes(self.nx, self.ny_global, int(slab[0]), int(slab[1]),
                                                        ctypes.byref(self.params), ctypes.byref(nbytes)))
        if not torch.cuda.is_available():
            raise TLBError(TLB_ECUDA, "no CUDA device; there is no CPU fallback")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.workspace = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) & ~255
        h = ctypes.c_void_p()
        self.h = None
        if slab is None:
            self._chk(self.lib.tlb_create(self.nx, self.ny_global, ctypes.byref(self.params), base, nbytes.value,
                                          self.stream.cuda_stream, ctypes.byref(h)))
        else:
            self._chk(self.lib.tlb_create_slab(self.nx, self.ny_global, int(slab[0]), int(slab[1]),
                                               ctypes.byref(self.params), base, nbytes.value,
                                               self.stream.cuda_stream, ctypes.byref(h)))
        self.h = h
        lay = (ctypes.c_int32 * 6)()
        self._chk(self.lib.tlb_slab_layout(self.h, lay))
        self.ny, self.own0, self.own1, self.y_off, self.halo_lo, self.halo_hi = (int(v) for v in lay)

    def _chk(self, rc):
        if rc != TLB_OK:
            msg = self.lib.tlb_error_string(rc).decode()
            if rc == TLB_ECUDA and getattr(self, "h", None):
                msg += ": " + self.lib.tlb_last_cuda_error(self.h).decode()
            raise TLBError(rc, msg)

    def close(self):
        if getattr(self, "h", None):
            self.lib.tlb_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dev(self, t, shape, dtype=None):
        torch = self.torch
        dtype = dtype or torch.float64
        t = torch.as_tensor(t)
        if t.device != self.device or t.dtype != dtype or not t.is_contiguous():
            # convert on the handle's stream: the kernels that read the temporary are enqueued there, so neither
            # the copy nor the caching allocator's reuse of the block can race with them
            with torch.cuda.stream(self.stream):
                t = t.to(device=self.device, dtype=dtype).contiguous()
        assert tuple(t.shape) == tuple(shape), (tuple(t.shape), shape)
        return t

    def _host(self, t, shape, dtype=None):
        torch = self.torch
        dtype = dtype or torch.float64
        t = torch.as_tensor(t)
        assert t.device.type == "cpu" and t.dtype == dtype and t.is_contiguous() and tuple(t.shape) == tuple(shape)
        return t

    def _new(self, *shape):
        return self.torch.empty(shape, dtype=self.torch.float64, device=self.device)

    # ---- the C calls -------------------------------------------------------------------------
    def init(self, seed):
        self._chk(self.lib.tlb_init(self.h, int(seed)))

    def set_solid(self, solid):
        s = self._dev(solid, (self.ny, self.nx), self.torch.uint8)
        self._chk(self.lib.tlb_set_solid(self.h, s.data_ptr()))

    def set_solid_host(self, solid):
        s = self._host(solid, (self.ny, self.nx), self.torch.uint8)
        self._chk(self.lib.tlb_set_solid_host(self.h, s.data_ptr()))

    def set_fields(self, rho_A, rho_B, T):
        a, b, t = (self._dev(v, (self.ny, self.nx)) for v in (rho_A, rho_B, T))
        self._chk(self.lib.tlb_set_fields(self.h, a.data_ptr(), b.data_ptr(), t.data_ptr()))

    def set_fields_host(self, rho_A, rho_B, T):
        a, b, t = (self._host(v, (self.ny, self.nx)) for v in (rho_A, rho_B, T))
        self._chk(self.lib.tlb_set_fields_host(self.h, a.data_ptr(), b.data_ptr(), t.data_ptr()))

    def set_populations(self, fA, fB, g):
        a, b, c = (self._dev(v, (9, self.ny, self.nx)) for v in (fA, fB, g))
        self._chk(self.lib.tlb_set_populations(self.h, a.data_ptr(), b.data_ptr(), c.data_ptr()))

    def get_populations(self):
        out = [self._new(9, self.ny, self.nx) for _ in range(3)]
        self._chk(self.lib.tlb_get_populations(self.h, *[o.data_ptr() for o in out]))
        return out

    def set_populations_host(self, fA, fB, g):
        a, b, c = (self._host(v, (9, self.ny, self.nx)) for v in (fA, fB, g))
        self._chk(self.lib.tlb_set_populations_host(self.h, a.data_ptr(), b.data_ptr(), c.data_ptr()))

    def get_populations_host(self, out=None):
        if out is None:
            out = [self.torch.empty((9, self.ny, self.nx), dtype=self.torch.float64) for _ in range(3)]
        a, b, c = (self._host(v, (9, self.ny, self.nx)) for v in out)
        self._chk(self.lib.tlb_get_populations_host(self.h, a.data_ptr(), b.data_ptr(), c.data_ptr()))
        return [a, b, c]

    def init_honeycomb(self, ndx, ndy, seed):
        self._chk(self.lib.tlb_init_honeycomb(self.h, int(ndx), int(ndy), int(seed)))

    def set_rough_walls(self, up, down, width, height, lam, alpha, asymmetric):
        r = TLBRoughWalls(alpha=float(alpha), up=int(up), down=int(down), width=int(width), height=int(height),
                          lam=int(lam), asymmetric=int(asymmetric))
        self._chk(self.lib.tlb_set_rough_walls(self.h, ctypes.byref(r)))

    def perturb_velocity(self, amplitude):
        self._chk(self.lib.tlb_perturb_velocity(self.h, float(amplitude)))

    def write_checkpoint(self, directory, index=0):
        self._chk(self.lib.tlb_write_checkpoint(self.h, os.fsencode(directory), int(index)))

    OUT_DENSITY, OUT_TEMPERATURE, OUT_VELOCITY, OUT_STRESS, OUT_ENERGY = 1, 2, 4, 8, 16

    def write_fields(self, directory, index=0, what=15, vtk=False):
        """The field files of Tables C.9 / C.10 (firstdensity.<i>.dat, ..., Pxy_av.<i>.dat; reading R31)."""
        self._chk(self.lib.tlb_write_fields(self.h, os.fsencode(directory), int(index), int(what), int(bool(vtk))))

    def read_checkpoint(self, directory, index=0):
        self._chk(self.lib.tlb_read_checkpoint(self.h, os.fsencode(directory), int(index)))

    def step(self, n=1):
        self._chk(self.lib.tlb_step(self.h, int(n)))

    def profile_step(self, n):
        """(fused_ms, boundary_ms): average duration of n back-to-back launches of each kernel (CUDA events on the
        stream); the state advances by one step."""
        a, b = ctypes.c_double(), ctypes.c_double()
        self._chk(self.lib.tlb_profile_step(self.h, int(n), ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def fields(self):
        rA, rB, T = self._new(self.ny, self.nx), self._new(self.ny, self.nx), self._new(self.ny, self.nx)
        u = self._new(2, self.ny, self.nx)
        self._chk(self.lib.tlb_fields(self.h, rA.data_ptr(), rB.data_ptr(), u.data_ptr(), T.data_ptr()))
        return rA, rB, u, T

    def fields_host(self, rho_A=None, rho_B=None, u=None, T=None):
        self._chk(self.lib.tlb_fields_host(self.h, _ptr(rho_A), _ptr(rho_B), _ptr(u), _ptr(T)))
        return rho_A, rho_B, u, T

    def observables(self):
        """dict(mass_A, mass_B, E, Nu) read back through tlb_observables_host."""
        out = (ctypes.c_double * 4)()
        self._chk(self.lib.tlb_observables_host(self.h, ctypes.cast(out, ctypes.c_void_p)))
        return dict(mass_A=out[0], mass_B=out[1], E=out[2], Nu=out[3])

    def x_average(self):
        """u_av[ny]: x-average of u_x^(H) over the fluid sites of each row (device tensor)."""
        out = self._new(self.ny)
        self._chk(self.lib.tlb_x_average(self.h, out.data_ptr()))
        return out

    def x_average_host(self, out=None):
        if out is None:
            out = self.torch.empty(self.ny, dtype=self.torch.float64)
        out = self._host(out, (self.ny,))
        self._chk(self.lib.tlb_x_average_host(self.h, out.data_ptr()))
        return out

    def observables_device(self, out4):
        self._chk(self.lib.tlb_observables(self.h, out4.data_ptr()))
        return out4

    def observable_sums(self, out6=None):
        """sums6 (device tensor): this handle's share of the six sums behind the observables."""
        out6 = self._new(6) if out6 is None else out6
        self._chk(self.lib.tlb_observable_sums(self.h, out6.data_ptr()))
        return out6

    def observables_from_sums(self, sums6):
        """dict(mass_A, mass_B, E, Nu) from (all-reduced) sums6 (device tensor)."""
        out = self._new(4)
        self._chk(self.lib.tlb_observables_from_sums(self.h, sums6.data_ptr(), out.data_ptr()))
        v = out.cpu().tolist()
        return dict(mass_A=v[0], mass_B=v[1], E=v[2], Nu=v[3])

    def stress_xy(self):
        """P_xy [ny][nx] (device tensor), reading R21."""
        out = self._new(self.ny, self.nx)
        self._chk(self.lib.tlb_stress_xy(self.h, out.data_ptr()))
        return out

    def stress_xy_host(self, out=None):
        if out is None:
            out = self.torch.empty((self.ny, self.nx), dtype=self.torch.float64)
        out = self._host(out, (self.ny, self.nx))
        self._chk(self.lib.tlb_stress_xy_host(self.h, out.data_ptr()))
        return out

    def x_average_stress(self):
        """Pxy_av[ny]: x-average of P_xy over the fluid sites of each row (device tensor)."""
        out = self._new(self.ny)
        self._chk(self.lib.tlb_x_average_stress(self.h, out.data_ptr()))
        return out

    def x_average_stress_host(self, out=None):
        if out is None:
            out = self.torch.empty(self.ny, dtype=self.torch.float64)
        out = self._host(out, (self.ny,))
        self._chk(self.lib.tlb_x_average_stress_host(self.h, out.data_ptr()))
        return out

    def droplets(self, B_th, max_droplets, want_labels=True):
        """(labels [ny][nx] int32 or None, n_droplets, stats [n][4]) as device tensors / int (section 2.4, R22)."""
        with self.torch.cuda.stream(self.stream):  # temporaries and read-backs on the stream the kernels run on
            torch = self.torch
            labels = torch.empty((self.ny, self.nx), dtype=torch.int32, device=self.device) if want_labels else None
            n = torch.zeros(1, dtype=torch.int32, device=self.device)
            stats = torch.zeros((max(1, max_droplets), 4), dtype=torch.float64, device=self.device)
            self._chk(self.lib.tlb_droplets(self.h, float(B_th), _ptr(labels), int(max_droplets), n.data_ptr(), stats.data_ptr()))
            k = int(n.item())
            return labels, k, stats[:min(k, max_droplets)]

    def droplets_host(self, B_th, max_droplets, want_labels=True):
        torch = self.torch
        labels = torch.empty((self.ny, self.nx), dtype=torch.int32) if want_labels else None
        n = torch.zeros(1, dtype=torch.int32)
        stats = torch.zeros((max(1, max_droplets), 4), dtype=torch.float64)
        self._chk(self.lib.tlb_droplets_host(self.h, float(B_th), _ptr(labels), int(max_droplets), n.data_ptr(), stats.data_ptr()))
        k = int(n.item())
        return labels, k, stats[:min(k, max_droplets)]

    # ---- droplet analysis, second stage (section 2.4, R23-R26): device tensors in, device tensors out
    def voronoi(self, centres):
        """colour [ny][nx] int32: index of the nearest centre; centres [n][2] float64 device tensor."""
        with self.torch.cuda.stream(self.stream):  # temporaries and read-backs on the stream the kernels run on
            torch = self.torch
            centres = centres.contiguous()
            colour = torch.empty((self.ny, self.nx), dtype=torch.int32, device=self.device)
            self._chk(self.lib.tlb_voronoi(self.h, _ptr(centres), int(centres.shape[0]), colour.data_ptr()))
            return colour

    def delaunay(self, colour, n, max_links=None):
        """(links [m][2] int32 sorted, n_links) from a colouring with n colours."""
        with self.torch.cuda.stream(self.stream):  # temporaries and read-backs on the stream the kernels run on
            torch = self.torch
            cap = int(max_links) if max_links is not None else 16 * max(1, int(n))
            links = torch.zeros((max(cap, 1), 2), dtype=torch.int32, device=self.device)
            nl = torch.zeros(1, dtype=torch.int32, device=self.device)
            self._chk(self.lib.tlb_delaunay(self.h, colour.data_ptr(), int(n), cap, nl.data_ptr(), links.data_ptr()))
            k = int(nl.item())
            return links[:max(0, min(k, cap))], k

    def droplet_match(self, colour_past, centres_now):
        with self.torch.cuda.stream(self.stream):  # temporaries and read-backs on the stream the kernels run on
            torch = self.torch
            centres_now = centres_now.contiguous()
            m = torch.zeros(max(1, int(centres_now.shape[0])), dtype=torch.int32, device=self.device)
            self._chk(self.lib.tlb_droplet_match(self.h, colour_past.data_ptr(), _ptr(centres_now), int(centres_now.shape[0]),
                                                 m.data_ptr()))
            return m[:int(centres_now.shape[0])]

    def droplet_displacements(self, centres_past, centres_now, map_now_to_past):
        """d_i = X_i(now) - X_map[i](past) [n_now][2] in minimum image (device tensor)."""
        with self.torch.cuda.stream(self.stream):
            torch = self.torch
            cp, cn, mp = centres_past.contiguous(), centres_now.contiguous(), map_now_to_past.contiguous()
            out = torch.zeros((max(1, int(cn.shape[0])), 2), dtype=torch.float64, device=self.device)
            self._chk(self.lib.tlb_droplet_displacements(self.h, _ptr(cp), _ptr(cn), _ptr(mp), int(cn.shape[0]), out.data_ptr()))
            return out[:int(cn.shape[0])]

    def t1_events(self, links_past, links_now, n_droplets, map_now_to_past=None, max_events=4096):
        """(events [e][4] int32 = (a, b, c, d): link a-b replaced by c-d, n_events)."""
        with self.torch.cuda.stream(self.stream):  # temporaries and read-backs on the stream the kernels run on
            torch = self.torch
            links_past, links_now = links_past.contiguous(), links_now.contiguous()
            ev = torch.zeros((max(1, max_events), 4), dtype=torch.int32, device=self.device)
            ne = torch.zeros(1, dtype=torch.int32, device=self.device)
            mp = map_now_to_past.contiguous() if map_now_to_past is not None else None
            self._chk(self.lib.tlb_t1_events(self.h, _ptr(links_past), int(links_past.shape[0]), _ptr(links_now),
                                             int(links_now.shape[0]), _ptr(mp), 0 if mp is None else int(mp.shape[0]),
                                             int(n_droplets), int(max_events), ne.data_ptr(), ev.data_ptr()))
            k = int(ne.item())
            return ev[:max(0, min(k, max_events))], k

    def droplet_nusselt(self, centres):
        """Nu_i of Eq. (25) [n] at the sites nearest to the centres [n][2]."""
        with self.torch.cuda.stream(self.stream):  # temporaries and read-backs on the stream the kernels run on
            torch = self.torch
            centres = centres.contiguous()
            nu = torch.zeros(max(1, int(centres.shape[0])), dtype=torch.float64, device=self.device)
            self._chk(self.lib.tlb_droplet_nusselt(self.h, _ptr(centres), int(centres.shape[0]), nu.data_ptr()))
            return nu[:int(centres.shape[0])]

    def seg_rows(self):
        return int(self.lib.tlb_seg_rows(self.h))

    # ---- y-slab stepping (tlb.h "Y-SLABS") ---------------------------------------------------
    def halo_buffer(self):
        """A device buffer of tlb_halo_bytes (one packed face)."""
        nb = ctypes.c_size_t()
        self._chk(self.lib.tlb_halo_bytes(self.h, ctypes.byref(nb)))
        return self.torch.empty(nb.value, dtype=self.torch.uint8, device=self.device)

    def slab_step_edges(self):
        self._chk(self.lib.tlb_slab_step_edges(self.h))

    def slab_step_interior(self):
        self._chk(self.lib.tlb_slab_step_interior(self.h))

    def slab_step_finish(self):
        self._chk(self.lib.tlb_slab_step_finish(self.h))

    def halo_region(self, face, which):
        """uint8 view (no copy) of the 3 owned rows next to `face` (which = 0) or of the halo rows beyond it (which = 1) in
        the population buffer that tlb_halo_pack / _unpack would address now."""
        p, nb = ctypes.c_void_p(), ctypes.c_size_t()
        self._chk(self.lib.tlb_halo_region(self.h, int(face), int(which), ctypes.byref(p), ctypes.byref(nb)))
        off = p.value - self.workspace.data_ptr()
        assert 0 <= off and off + nb.value <= self.workspace.numel()
        return self.workspace[off:off + nb.value]

    def halo_pack(self, face, buf):
        self._chk(self.lib.tlb_halo_pack(self.h, int(face), buf.data_ptr()))

    def halo_unpack(self, face, buf):
        self._chk(self.lib.tlb_halo_unpack(self.h, int(face), buf.data_ptr()))

    def launch_count(self):
        return int(self.lib.tlb_launch_count(self.h))


def params_from_config(cfg):
    """TLBParams for a workload dict of inputs.config()."""
    pw, ph, pp = cfg["posts"]
    kw = dict(cfg["params"])
    kw.update(cfg["init"])
    kw.update(post_w=pw, post_h=ph, post_period=pp)
    return default_params(**kw)
