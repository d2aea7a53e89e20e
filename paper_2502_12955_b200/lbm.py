"""Thin Python binding of the C-ABI library (include/lbm.h -> paper_2502_12955_b200/liblbm.so).

Argument marshalling only: every step of the lattice Boltzmann path runs in the CUDA kernels of
csrc/.  PyTorch supplies device memory (the workspace and the output buffers) and the stream.
There is no CPU fallback: if liblbm.so is missing the import of the library fails loudly, and
lbm_create fails when no CUDA device is usable.  Nothing here imports oracle/.
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "liblbm.so")

D2Q9, D3Q19 = 0, 1
BGK, SC1, SC2, SC2_ADE, BGK_T = 0, 1, 2, 3, 4
LATTICES = {"D2Q9": D2Q9, "D3Q19": D3Q19}
MODELS = {"BGK": BGK, "SC1": SC1, "SC2": SC2, "SC2_ADE": SC2_ADE, "BGK_T": BGK_T}
INITS = {"REST": 0, "TAYLOR_GREEN": 1, "DROPLET": 2, "UNIFORM_NOISE": 3, "RANDOM_DROPLETS": 4}
OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, -1, -2, -3, -4
PATHS = {"register": 0, "pipeline": 1}

# every symbol include/lbm.h declares (tests check that the library exports each one)
SYMBOLS = ("lbm_workspace_bytes", "lbm_create", "lbm_init_from_seed", "lbm_step", "lbm_get_macros",
           "lbm_get_force", "lbm_population_count", "lbm_get_populations", "lbm_set_populations",
           "lbm_run_host", "lbm_set_path", "lbm_get_path", "lbm_set_mask", "lbm_tile_schedule", "lbm_tile_tickets", "lbm_check", "lbm_static_scratch_bytes", "lbm_step_static", "lbm_time", "lbm_launch_count", "lbm_kernel_timing", "lbm_kernel_time_ms", "lbm_lattice_table", "lbm_destroy",
           "lbm_last_error")


class LbmParams(C.Structure):
    """struct lbm_params of include/lbm.h, field for field."""
    _fields_ = [
        ("struct_size", C.c_uint32), ("precision", C.c_int32),
        ("tau", C.c_double * 2), ("tau_c", C.c_double),
        ("G", (C.c_double * 2) * 2),
        ("psi_kind", C.c_int32), ("forcing", C.c_int32),
        ("rho0_psi", C.c_double), ("force", C.c_double * 3),
        ("bc", C.c_int32 * 3), ("init_kind", C.c_int32),
        ("k_react", C.c_double), ("w0_scalar", C.c_double),
        ("rho_init", C.c_double * 2), ("c_init", C.c_double),
        ("rho_in", C.c_double), ("rho_out", C.c_double), ("radius", C.c_double), ("width", C.c_double),
        ("noise_amp", C.c_double), ("u0", C.c_double), ("rmin", C.c_double), ("rmax", C.c_double),
        ("vol_frac", C.c_double), ("G_ads", C.c_double * 2), ("rho_wall", C.c_double), ("wall_u", ((C.c_double * 3) * 2) * 3),
        ("tau_s", C.c_double), ("rho_solid", C.c_double),
        ("workspace", C.c_void_p), ("stream", C.c_void_p),
    ]


class LbmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("lbm error %d: %s" % (code, msg))
        self.code = code


_lib = None


def lib():
    """Load liblbm.so (built in-tree by paper_2502_12955_b200/build.py).  No fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s is missing: run `python -m paper_2502_12955_b200.build` (needs nvcc); "
                          "there is no CPU fallback" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    P = C.POINTER(LbmParams)
    L.lbm_workspace_bytes.restype = C.c_size_t
    L.lbm_workspace_bytes.argtypes = [C.c_int] * 5 + [P]
    L.lbm_create.restype = C.c_void_p
    L.lbm_create.argtypes = [C.c_int] * 5 + [P]
    L.lbm_init_from_seed.argtypes = [C.c_void_p, C.c_uint64]
    L.lbm_step.argtypes = [C.c_void_p, C.c_int]
    L.lbm_get_macros.argtypes = [C.c_void_p] * 5
    L.lbm_get_force.argtypes = [C.c_void_p, C.c_void_p]
    L.lbm_population_count.restype = C.c_size_t
    L.lbm_population_count.argtypes = [C.c_void_p]
    L.lbm_get_populations.argtypes = [C.c_void_p, C.c_void_p]
    L.lbm_set_populations.argtypes = [C.c_void_p, C.c_void_p]
    L.lbm_run_host.argtypes = [C.c_void_p, C.c_void_p, C.c_int] + [C.c_void_p] * 4
    L.lbm_tile_tickets.argtypes = [C.c_int] * 8 + [C.c_void_p, C.c_size_t, C.POINTER(C.c_size_t)]
    L.lbm_static_scratch_bytes.restype = C.c_size_t
    L.lbm_static_scratch_bytes.argtypes = []
    L.lbm_step_static.argtypes = [C.c_int] * 5 + [P, C.c_void_p, C.c_int]
    L.lbm_set_path.argtypes = [C.c_void_p, C.c_int, C.c_int]
    L.lbm_get_path.argtypes = [C.c_void_p]
    L.lbm_set_mask.argtypes = [C.c_void_p, C.c_void_p]
    L.lbm_tile_schedule.argtypes = [C.c_int] * 6 + [C.c_void_p, C.c_size_t, C.POINTER(C.c_size_t), C.POINTER(C.c_int)]
    L.lbm_check.argtypes = [C.c_void_p]
    L.lbm_time.restype = C.c_int64
    L.lbm_time.argtypes = [C.c_void_p]
    L.lbm_launch_count.restype = C.c_int64
    L.lbm_launch_count.argtypes = [C.c_void_p]
    L.lbm_kernel_timing.argtypes = [C.c_void_p, C.c_int]
    L.lbm_kernel_time_ms.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
    L.lbm_lattice_table.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_int), C.c_void_p, C.c_void_p, C.c_void_p]
    L.lbm_destroy.argtypes = [C.c_void_p]
    L.lbm_last_error.restype = C.c_char_p
    _lib = L
    return L


def last_error():
    return lib().lbm_last_error().decode()


def make_params(**kw):
    """Fill an LbmParams from keyword arguments (the keys of workloads.py's dictionaries)."""
    p = LbmParams()
    p.struct_size = C.sizeof(LbmParams)
    p.precision = int(kw.get("precision", 64))
    tau = kw.get("tau", (1.0, 1.0))
    if not isinstance(tau, (tuple, list)):
        tau = (tau, tau)
    p.tau[0], p.tau[1] = float(tau[0]), float(tau[1])
    p.tau_c = float(kw.get("tau_c", 1.0))
    G = kw.get("G", ((0.0, 0.0), (0.0, 0.0)))
    for s in range(2):
        for t in range(2):
            p.G[s][t] = float(G[s][t])
    p.psi_kind = int(kw.get("psi_kind", 0))
    p.forcing = int(kw.get("forcing", 0))
    p.rho0_psi = float(kw.get("rho0_psi", 1.0))
    for a, v in enumerate(kw.get("force", (0.0, 0.0, 0.0))):
        p.force[a] = float(v)
    for a, v in enumerate(kw.get("bc", (0, 0, 0))):
        p.bc[a] = int(v)
    init = kw.get("init_kind", "REST")
    p.init_kind = INITS[init] if isinstance(init, str) else int(init)
    p.k_react = float(kw.get("k_react", 0.0))
    p.w0_scalar = float(kw.get("w0_scalar", 0.0))
    ri = kw.get("rho_init", (1.0, 1.0))
    if not isinstance(ri, (tuple, list)):
        ri = (ri, ri)
    p.rho_init[0], p.rho_init[1] = float(ri[0]), float(ri[1])
    p.c_init = float(kw.get("c_init", 0.0))
    for k, dflt in (("rho_in", 1.0), ("rho_out", 1.0), ("radius", 0.0), ("width", 3.0), ("noise_amp", 0.0),
                    ("u0", 0.0), ("rmin", 0.0), ("rmax", 0.0), ("vol_frac", 0.0)):
        setattr(p, k, float(kw.get(k, dflt)))
    ga = kw.get("G_ads", (0.0, 0.0))
    p.G_ads[0], p.G_ads[1] = float(ga[0]), float(ga[1])
    p.rho_wall = float(kw.get("rho_wall", 0.0))
    p.tau_s = float(kw.get("tau_s", 0.0))
    p.rho_solid = float(kw.get("rho_solid", 1.0))
    for (axis, side), v in kw.get("wall_u", {}).items():      # {(axis, side): (ux, uy, uz)}, side 0 = low, 1 = high face
        for a in range(3):
            p.wall_u[axis][side][a] = float(v[a])
    p.workspace = None
    p.stream = None
    return p


def tile_schedule(nm, ns, rows_per_pencil, wrap_m=True, wrap_s=True, delay_rows=0):
    """The resident-tile kernel's row schedule as an (n, 3) int32 array of (kind, m, s), and the number of psi rows
    that wait for another pencil; host-only call (kind 0: step of the row, 1: psi of the next time level)."""
    import numpy as np
    L = lib()
    n = C.c_size_t(0)
    lead = C.c_int(0)
    rc = L.lbm_tile_schedule(nm, ns, rows_per_pencil, int(wrap_m), int(wrap_s), int(delay_rows), None, 0, C.byref(n), C.byref(lead))
    if rc != 0:
        raise LbmError(rc, last_error())
    out = np.zeros((n.value, 3), np.int32)
    rc = L.lbm_tile_schedule(nm, ns, rows_per_pencil, int(wrap_m), int(wrap_s), int(delay_rows), out.ctypes.data, n.value, C.byref(n), C.byref(lead))
    if rc != 0:
        raise LbmError(rc, last_error())
    return out, lead.value


def tile_tickets(nm, ns, nxs, rows_per_pencil, wrap_m=True, wrap_s=True, delay_rows=0, three_d=True):
    """The resident-tile kernel's tickets as an (n, 8) int32 array (sx, sy, sz, sv, px, py, pz, pv); host-only call."""
    import numpy as np
    L = lib()
    n = C.c_size_t(0)
    args = (int(nm), int(ns), int(nxs), int(rows_per_pencil), int(wrap_m), int(wrap_s), int(delay_rows), int(three_d))
    rc = L.lbm_tile_tickets(*args, None, 0, C.byref(n))
    if rc != 0:
        raise LbmError(rc, last_error())
    out = np.zeros((n.value, 8), np.int32)
    rc = L.lbm_tile_tickets(*args, out.ctypes.data, n.value, C.byref(n))
    if rc != 0:
        raise LbmError(rc, last_error())
    return out


def static_scratch_bytes():
    return int(lib().lbm_static_scratch_bytes())


def step_static(nx, ny, nz, lattice, model, f, n, stream=None, **params):
    """lbm_step_static: n (even) steps of a Shan-Chen model in place on the device tensor f of canonical populations,
    with the psi field in the library's static device array -- no allocation (include/lbm.h).  Marshalling only."""
    L = lib()
    p = make_params(**params)
    p.stream = stream
    lat = LATTICES[lattice] if isinstance(lattice, str) else int(lattice)
    mod = MODELS[model] if isinstance(model, str) else int(model)
    rc = L.lbm_step_static(int(nx), int(ny), int(nz), lat, mod, C.byref(p), f.data_ptr(), int(n))
    if rc != 0:
        raise LbmError(rc, last_error())


def lattice_table(lattice, kind=0):
    """(c[Q,3], w[Q], opp[Q]) as the kernels use them; host-only call."""
    import numpy as np
    L = lib()
    Q = C.c_int(0)
    c = np.zeros((19, 3), np.int32)
    w = np.zeros(19, np.float64)
    opp = np.zeros(19, np.int32)
    rc = L.lbm_lattice_table(LATTICES[lattice] if isinstance(lattice, str) else lattice, kind, C.byref(Q),
                             c.ctypes.data, w.ctypes.data, opp.ctypes.data)
    if rc != 0:
        raise LbmError(rc, last_error())
    return c[:Q.value].copy(), w[:Q.value].copy(), opp[:Q.value].copy()


class LBM:
    """One library context.  Field arguments and results are torch CUDA tensors in the context
    precision; `device` is a torch device, `stream` a torch.cuda.Stream (default: current)."""

    def __init__(self, nx, ny, nz, lattice, model, device="cuda:0", stream=None, **params):
        import torch
        self.torch = torch
        self.L = lib()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.lattice = LATTICES[lattice] if isinstance(lattice, str) else int(lattice)
        self.model = MODELS[model] if isinstance(model, str) else int(model)
        self.p = make_params(**params)
        self.dtype = torch.float64 if self.p.precision == 64 else torch.float32
        self.S = 2 if self.model in (SC2, SC2_ADE) else 1
        self.d = 3 if self.lattice == D3Q19 else 2
        self.Q = 19 if self.lattice == D3Q19 else 9
        self.Qs = 7 if self.lattice == D3Q19 else 5
        self.has_scalar = self.model in (SC2_ADE, BGK_T)      # a second lattice with a C / eps output
        self.N = self.nx * self.ny * self.nz
        self.h = None
        self.device = torch.device(device)
        nbytes = self.L.lbm_workspace_bytes(self.nx, self.ny, self.nz, self.lattice, self.model, C.byref(self.p))
        if nbytes == 0:
            raise LbmError(EINVAL, last_error())
        if not torch.cuda.is_available():
            raise LbmError(ECUDA, "no CUDA device: this library has no CPU path")
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        with torch.cuda.device(self.device):
            # device memory comes from torch (caching allocator returns 512-byte aligned blocks)
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.p.workspace = self.workspace.data_ptr()
            self.p.stream = self.stream.cuda_stream
            self.h = self.L.lbm_create(self.nx, self.ny, self.nz, self.lattice, self.model, C.byref(self.p))
        if not self.h:
            raise LbmError(EINVAL, last_error())

    def _chk(self, rc):
        if rc != 0:
            raise LbmError(rc, last_error())

    def _new(self, *shape):
        return self.torch.empty(shape, dtype=self.dtype, device=self.device)

    @staticmethod
    def _ptr(t):
        return None if t is None else t.data_ptr()

    def init_from_seed(self, seed):
        self._chk(self.L.lbm_init_from_seed(self.h, int(seed)))

    def step(self, n=1):
        self._chk(self.L.lbm_step(self.h, int(n)))

    def get_macros(self, rho=True, u=True, phi=True, C_=True):
        """dict of device tensors rho (S,N), u (d,N), phi (N), C (N or None)"""
        out = {"rho": self._new(self.S, self.N) if rho else None,
               "u": self._new(self.d, self.N) if u else None,
               "phi": self._new(self.N) if phi else None,
               "C": self._new(self.N) if (C_ and self.has_scalar) else None}
        self._chk(self.L.lbm_get_macros(self.h, self._ptr(out["rho"]), self._ptr(out["u"]), self._ptr(out["phi"]),
                                        self._ptr(out["C"])))
        return out

    def get_force(self):
        F = self._new(self.S, self.d, self.N)
        self._chk(self.L.lbm_get_force(self.h, F.data_ptr()))
        return F

    def population_count(self):
        return int(self.L.lbm_population_count(self.h))

    def get_populations(self):
        f = self._new(self.population_count())
        self._chk(self.L.lbm_get_populations(self.h, f.data_ptr()))
        return f

    def set_populations(self, f):
        f = f.to(device=self.device, dtype=self.dtype).contiguous()
        assert f.numel() == self.population_count()
        self._chk(self.L.lbm_set_populations(self.h, f.data_ptr()))
        self.stream.synchronize()   # f may be a temporary

    def run_host(self, f_in, n, rho=None, u=None, phi=None, C_=None):
        """lbm_run_host: host (numpy or CPU torch, ideally pinned) buffers in and out."""
        def hp(a):
            if a is None:
                return None
            return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
        self._chk(self.L.lbm_run_host(self.h, hp(f_in), int(n), hp(rho), hp(u), hp(phi), hp(C_)))

    def time(self):
        return int(self.L.lbm_time(self.h))

    def launch_count(self):
        return int(self.L.lbm_launch_count(self.h))

    def kernel_timing(self, enable):
        self._chk(self.L.lbm_kernel_timing(self.h, 1 if enable else 0))

    def kernel_time_ms(self, kind):
        """(summed device ms, launches) of kind 0 = fused step kernel, 1 = psi pass"""
        ms, n = C.c_double(0.0), C.c_int64(0)
        self._chk(self.L.lbm_kernel_time_ms(self.h, int(kind), C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def set_path(self, path, rows_per_pencil=0):
        """which kernels step() launches: "register" or "pipeline" (Shan-Chen models; include/lbm.h)"""
        path = PATHS[path] if isinstance(path, str) else int(path)
        self._chk(self.L.lbm_set_path(self.h, path, int(rows_per_pencil)))

    def set_mask(self, mask):
        """solid-node mask (N values, non-zero = solid; any array-like or tensor) or None; kept alive here"""
        if mask is None:
            self._chk(self.L.lbm_set_mask(self.h, None))
            self._mask = None
            return
        m = self.torch.as_tensor(mask).to(device=self.device, dtype=self.torch.uint8).contiguous().reshape(-1)
        assert m.numel() == self.N
        self._chk(self.L.lbm_set_mask(self.h, m.data_ptr()))
        self._mask = m

    def get_path(self):
        return {v: k for k, v in PATHS.items()}[self.L.lbm_get_path(self.h)]

    def check(self):
        """synchronise and raise on deferred device-side errors"""
        self._chk(self.L.lbm_check(self.h))

    def synchronize(self):
        self.stream.synchronize()

    def close(self):
        if self.h:
            self.L.lbm_destroy(self.h)
            self.h = None
        self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
