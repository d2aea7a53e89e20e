"""ctypes binding of the CPU oracle (oracle/libref_lbm.so).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It imports nothing from paper_2502_12955_b200.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))

D2Q9, D3Q19 = 0, 1
BGK, SC1, SC2, SC2_ADE, BGK_T = 0, 1, 2, 3, 4
INIT_REST, INIT_TAYLOR_GREEN, INIT_DROPLET, INIT_UNIFORM_NOISE, INIT_RANDOM_DROPLETS = 0, 1, 2, 3, 4
LATTICES = {"D2Q9": D2Q9, "D3Q19": D3Q19}
MODELS = {"BGK": BGK, "SC1": SC1, "SC2": SC2, "SC2_ADE": SC2_ADE, "BGK_T": BGK_T}
INITS = {"REST": INIT_REST, "TAYLOR_GREEN": INIT_TAYLOR_GREEN, "DROPLET": INIT_DROPLET,
         "UNIFORM_NOISE": INIT_UNIFORM_NOISE, "RANDOM_DROPLETS": INIT_RANDOM_DROPLETS}


class RefParams(C.Structure):
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
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        from . import build as _b  # noqa
        path = _b.build()
        L = C.CDLL(path)
        L.ref_create.restype = C.c_void_p
        L.ref_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(RefParams)]
        L.ref_init_from_seed.argtypes = [C.c_void_p, C.c_uint64]
        L.ref_step.argtypes = [C.c_void_p, C.c_int]
        L.ref_get_macros.argtypes = [C.c_void_p] + [C.c_void_p] * 4
        L.ref_get_force.argtypes = [C.c_void_p, C.c_void_p]
        L.ref_set_mask.argtypes = [C.c_void_p, C.c_void_p]
        L.ref_get_populations.argtypes = [C.c_void_p, C.c_void_p]
        L.ref_set_populations.argtypes = [C.c_void_p, C.c_void_p]
        L.ref_population_count.restype = C.c_size_t
        L.ref_population_count.argtypes = [C.c_void_p]
        L.ref_destroy.argtypes = [C.c_void_p]
        L.ref_last_error.restype = C.c_char_p
        L.ref_lattice_table.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_int), C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def make_params(**kw):
    """Fill a RefParams from keyword arguments (the keys of workloads.py's dictionaries)."""
    p = RefParams()
    p.struct_size = C.sizeof(RefParams)
    p.precision = int(kw.get("precision", 64))
    tau = kw.get("tau", (1.0, 1.0))
    if np.isscalar(tau):
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
    if np.isscalar(ri):
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
    for (axis, side), v in kw.get("wall_u", {}).items():      # {(axis, side): (ux, uy, uz)}, side 0 = low face, 1 = high face
        for a in range(3):
            p.wall_u[axis][side][a] = float(v[a])
    return p


class RefLBM:
    """One oracle context; all arrays are host numpy arrays in the context precision."""

    def __init__(self, nx, ny, nz, lattice, model, **params):
        self.L = lib()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.lattice = LATTICES[lattice] if isinstance(lattice, str) else int(lattice)
        self.model = MODELS[model] if isinstance(model, str) else int(model)
        self.p = make_params(**params)
        self.dtype = np.float64 if self.p.precision == 64 else np.float32
        self.S = 2 if self.model in (SC2, SC2_ADE) else 1
        self.d = 3 if self.lattice == D3Q19 else 2
        self.Q = 19 if self.lattice == D3Q19 else 9
        self.Qs = 7 if self.lattice == D3Q19 else 5
        self.has_scalar = self.model == SC2_ADE
        self.has_thermal = self.model == BGK_T
        self.N = self.nx * self.ny * self.nz
        self.h = self.L.ref_create(self.nx, self.ny, self.nz, self.lattice, self.model, C.byref(self.p))
        if not self.h:
            raise ValueError("ref_create: " + self.L.ref_last_error().decode())

    def _chk(self, rc):
        if rc != 0:
            raise RuntimeError("oracle: " + self.L.ref_last_error().decode())

    def init_from_seed(self, seed):
        self._chk(self.L.ref_init_from_seed(self.h, int(seed)))

    def step(self, n):
        self._chk(self.L.ref_step(self.h, int(n)))

    def get_macros(self):
        """returns dict rho (S,N), u (d,N), phi (N), C (N) or None"""
        rho = np.empty((self.S, self.N), self.dtype)
        u = np.empty((self.d, self.N), self.dtype)
        phi = np.empty(self.N, self.dtype)
        Cc = np.empty(self.N, self.dtype) if (self.has_scalar or self.has_thermal) else None
        self._chk(self.L.ref_get_macros(self.h, rho.ctypes.data, u.ctypes.data, phi.ctypes.data,
                                        Cc.ctypes.data if Cc is not None else None))
        return {"rho": rho, "u": u, "phi": phi, "C": Cc}

    def get_force(self):
        F = np.empty((self.S, self.d, self.N), self.dtype)
        self._chk(self.L.ref_get_force(self.h, F.ctypes.data))
        return F

    def set_mask(self, mask):
        """solid-node mask: N values, non-zero = solid; None clears it"""
        if mask is None:
            self._chk(self.L.ref_set_mask(self.h, None))
        else:
            m = np.ascontiguousarray(mask, dtype=np.uint8).ravel()
            assert m.size == self.N
            self._chk(self.L.ref_set_mask(self.h, m.ctypes.data))

    def population_count(self):
        return int(self.L.ref_population_count(self.h))

    def get_populations(self):
        f = np.empty(self.population_count(), self.dtype)
        self._chk(self.L.ref_get_populations(self.h, f.ctypes.data))
        return f

    def set_populations(self, f):
        f = np.ascontiguousarray(f, dtype=self.dtype)
        assert f.size == self.population_count()
        self._chk(self.L.ref_set_populations(self.h, f.ctypes.data))

    def split_populations(self, f):
        """canonical vector -> (f[S,Q,N], h[Qs,N] or None)"""
        nf = self.S * self.Q * self.N
        ff = f[:nf].reshape(self.S, self.Q, self.N)
        hh = f[nf:].reshape(self.Qs, self.N) if self.has_scalar else (f[nf:].reshape(self.Q, self.N) if self.has_thermal else None)
        return ff, hh

    def close(self):
        if self.h:
            self.L.ref_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lattice_table(lattice, kind=0):
    L = lib()
    Q = C.c_int(0)
    c = np.zeros((19, 3), np.int32)
    w = np.zeros(19, np.float64)
    L.ref_lattice_table(LATTICES[lattice] if isinstance(lattice, str) else lattice, kind, C.byref(Q),
                        c.ctypes.data, w.ctypes.data)
    return c[:Q.value].copy(), w[:Q.value].copy()
